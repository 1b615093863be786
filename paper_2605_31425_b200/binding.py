"""Thin ctypes binding of libmeb_b200.so (include/meb.h).  Argument marshalling ONLY:
every step of the path runs in the CUDA kernels of the library.  PyTorch is used for device
memory (``tensor.data_ptr()``) and the current stream, nothing else.

The library is mandatory: ``load()`` raises if it is missing (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmeb_b200.so")

MEB_OK = 0
MEB_W_NOT_CONVERGED = 1
MEB_E_ARG, MEB_E_INPUT, MEB_E_ALLOC, MEB_E_CUDA, MEB_E_CAPACITY = -1, -2, -3, -4, -5
MEB_FP64, MEB_FP32 = 0, 1
MEB_MODE_FP64, MEB_MODE_MIXED = 0, 1
MEB_EVAL_NSCALARS = 16
OPT = dict(STEPPED=0, NO_SMALL=1, NO_ABORT=2, NO_FUSED_SCREEN=3)
PASS = dict(INGEST=0, EVAL_FP64=1, EVAL_FP32=2, SCREEN=3, FEAS=4, EVAL_REDUCED=5)
EV = dict(PSI=0, SUM_UPLUS=1, SUM_PROJ2=2, SUM_DMULT2=3, N_B1=4, N_B3=5, MAX_PFEAS=6, MAX_COMPL=7,
          MAX_DFEAS=8, SUM_RHO=9, NORM_SUM_VPLUS=10, N_ACTIVE=11)

EXPORTS = [
    "meb_create", "meb_destroy", "meb_strerror", "meb_last_cuda_error", "meb_default_params",
    "meb_version", "meb_solve", "meb_solve_host", "meb_ingest", "meb_eval_alm", "meb_hvp",
    "meb_dense_hessian", "meb_update_multipliers", "meb_screen_compact", "meb_feasibility_check",
    "meb_feasibility_max_static",
    "meb_last_pass_info", "meb_set_pass_timing", "meb_solve_batch", "meb_set_option", "meb_eval_alm_multi",
    "meb_solve_sharded", "meb_shard_record_doubles",
]
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64)


class meb_params(C.Structure):
    _fields_ = [("rho", C.c_double), ("sigma0", C.c_double), ("kappa", C.c_double),
                ("sigma_max", C.c_double), ("tau", C.c_double), ("armijo_mu", C.c_double),
                ("tol_lo", C.c_double), ("tol_red_factor", C.c_double),
                ("armijo_max_halvings", C.c_int32), ("cg_max", C.c_int32), ("dense_d_max", C.c_int32),
                ("inner_max", C.c_int32), ("outer_max", C.c_int32), ("max_rounds", C.c_int32),
                ("sample_rows", C.c_int32), ("outer_max_lo", C.c_int32), ("armijo_shrink_min", C.c_double),
                ("armijo_multi", C.c_int32), ("ag_outer", C.c_int32), ("sigma_carry", C.c_double)]


class meb_stats(C.Structure):
    _fields_ = [("converged", C.c_int32), ("outer_iters", C.c_int32), ("newton_iters", C.c_int32),
                ("cg_iters", C.c_int32), ("passes_fp64_full", C.c_int32), ("passes_fp32_full", C.c_int32),
                ("passes_reduced", C.c_int32), ("rounds", C.c_int32), ("n_reduced", C.c_int64),
                ("n_support", C.c_int64), ("kkt", C.c_double), ("kkt_terms", C.c_double * 5),
                ("delta_max", C.c_double), ("radius_alg", C.c_double), ("length_scale", C.c_double),
                ("ms_total", C.c_double), ("ms_phase_lo", C.c_double), ("ms_phase_hi", C.c_double),
                ("ms_check", C.c_double), ("bytes_streamed", C.c_double),
                ("pass_ms", C.c_double * 8), ("pass_bytes", C.c_double * 8), ("pass_count", C.c_int32 * 8),
                ("kernel_launches", C.c_int64), ("passes_cut", C.c_int32), ("trials_skipped", C.c_int32),
                ("pass_ev_ms", C.c_double * 8), ("pass_ev_bytes", C.c_double * 8), ("pass_ev_count", C.c_int32 * 8),
                ("ag_iters", C.c_int32), ("reserved0", C.c_int32)]

    def as_dict(self):
        out = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            out[name] = list(v) if hasattr(v, "__len__") else v
        return out


class MebError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: {strerror(code)} (code {code})")
        self.code = code


_lib = None


def load():
    """Load libmeb_b200.so; raise loudly if it has not been built (no fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with paper_2605_31425_b200/build.sh "
            "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl, flt = C.c_void_p, C.c_int32, C.c_int64, C.c_double, C.c_float
    lib.meb_create.argtypes = [C.POINTER(vp), C.c_int, vp, i64, i32]
    lib.meb_destroy.argtypes = [vp]
    lib.meb_strerror.argtypes = [C.c_int]
    lib.meb_strerror.restype = C.c_char_p
    lib.meb_last_cuda_error.argtypes = [vp]
    lib.meb_default_params.argtypes = [C.POINTER(meb_params)]
    lib.meb_default_params.restype = None
    lib.meb_set_pass_timing.argtypes = [vp, C.c_int]
    lib.meb_set_option.argtypes = [vp, C.c_int, C.c_int]
    lib.meb_last_pass_info.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]
    solve_args = [vp, i64, i32, vp, i64, vp, dbl, C.c_int, C.POINTER(meb_params), vp, C.POINTER(dbl),
                  C.POINTER(meb_stats)]
    lib.meb_solve.argtypes = solve_args
    lib.meb_solve_host.argtypes = solve_args
    lib.meb_solve_batch.argtypes = [vp, i32, vp, i32, vp, i64, vp, dbl, C.POINTER(meb_params), vp, vp, vp, vp]
    lib.meb_shard_record_doubles.argtypes = [i32]
    lib.meb_shard_record_doubles.restype = i64
    lib.meb_solve_sharded.argtypes = [vp, i32, i32, i64, i64, i64, i32, vp, i64, vp, dbl, C.c_int, C.POINTER(meb_params),
                                      vp, vp, i64, ALLGATHER_FN, vp, vp, C.POINTER(dbl), C.POINTER(meb_stats)]
    lib.meb_ingest.argtypes = [vp, i64, i32, vp, i64, vp, i32, vp, vp, vp, i64, vp]
    prob = [vp, C.c_int, i64, i32, vp, i64, vp, vp, vp, vp, i64]
    lib.meb_eval_alm.argtypes = prob + [vp, vp, dbl, dbl, vp, vp, vp, vp, vp, vp, vp]
    lib.meb_eval_alm_multi.argtypes = prob + [vp, vp, dbl, dbl, vp, i32, vp, vp, vp, vp]
    lib.meb_hvp.argtypes = prob + [vp, dbl, dbl, vp, vp]
    lib.meb_dense_hessian.argtypes = prob + [vp, dbl, dbl, vp]
    lib.meb_update_multipliers.argtypes = prob + [vp, dbl, vp, vp, vp, i64, i64, C.POINTER(i64), C.POINTER(dbl)]
    lib.meb_screen_compact.argtypes = [vp, i64, i32, vp, i64, vp, flt, vp, flt, vp, i64, C.POINTER(i64), vp,
                                       C.c_int]
    lib.meb_feasibility_max_static.argtypes = [vp, i64, i32, vp, i64, vp, dbl, vp, vp]
    lib.meb_feasibility_check.argtypes = [vp, i64, i32, vp, i64, vp, dbl, vp, dbl, vp, C.POINTER(dbl),
                                          C.POINTER(i32), vp, i64, C.POINTER(i64)]
    for name in EXPORTS:
        fn = getattr(lib, name)
        if name not in ("meb_strerror", "meb_default_params", "meb_shard_record_doubles"):
            fn.restype = C.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().meb_strerror(int(code)).decode()


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _check(code, what, allow=(MEB_OK,)):
    if code not in allow:
        raise MebError(code, what)
    return code


def _dt(prec):
    return torch.float64 if prec == MEB_FP64 else torch.float32


def _problem(prec, Cm, R, U, v_slot, Vrows):
    assert Cm.is_cuda and Cm.dtype == _dt(prec) and Cm.dim() == 2 and Cm.stride(1) == 1
    m, d = Cm.shape
    ld = Cm.stride(0)
    for t in (R, U):
        assert t is None or (t.is_cuda and t.dtype == _dt(prec) and t.is_contiguous() and t.numel() == m)
    ldv = 0
    if v_slot is not None:
        assert v_slot.dtype == torch.int32 and v_slot.is_contiguous() and v_slot.numel() == m
        assert Vrows is not None and Vrows.dtype == _dt(prec) and Vrows.stride(1) == 1
        ldv = Vrows.stride(0)
    return m, d, ld, ldv


def meb_default_params() -> meb_params:
    p = meb_params()
    load().meb_default_params(C.byref(p))
    return p


class Context:
    """Owns a ``meb_ctx`` (workspace for problems up to m_max x d_max) on the current CUDA device."""

    def __init__(self, m_max: int, d_max: int, device: int | None = None, stream=None):
        lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2605_31425_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.cuda.current_device() if device is None else int(device)
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        self._stream = s
        h = C.c_void_p()
        _check(lib.meb_create(C.byref(h), self.device, C.c_void_p(s.cuda_stream), int(m_max), int(d_max)),
               "meb_create")
        self.h = h
        self.m_max, self.d_max = int(m_max), int(d_max)

    def close(self):
        if getattr(self, "h", None):
            load().meb_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


def meb_set_pass_timing(ctx: Context, on: bool):
    _check(load().meb_set_pass_timing(ctx.h, int(bool(on))), "meb_set_pass_timing")


def meb_set_option(ctx: Context, option: int, value: bool):
    _check(load().meb_set_option(ctx.h, int(option), int(bool(value))), "meb_set_option")


def meb_last_pass_info(ctx: Context):
    ms, by = C.c_double(), C.c_double()
    _check(load().meb_last_pass_info(ctx.h, C.byref(ms), C.byref(by)), "meb_last_pass_info")
    return ms.value, by.value


def meb_solve(ctx: Context, centers, radii, tol=1e-8, precision_mode=MEB_MODE_FP64, params=None,
              allow_not_converged=False):
    """centers (m, d) float64 CUDA tensor (row stride >= d), radii (m,) or None.
    Returns (center numpy-like CPU tensor (d,), radius float, stats dict)."""
    assert centers.is_cuda and centers.dtype == torch.float64 and centers.stride(1) == 1
    m, d = centers.shape
    out_c = torch.empty(d, dtype=torch.float64)
    out_r = C.c_double()
    st = meb_stats()
    code = load().meb_solve(ctx.h, m, d, _ptr(centers), centers.stride(0), _ptr(radii), float(tol),
                            int(precision_mode), None if params is None else C.byref(params),
                            C.c_void_p(out_c.data_ptr()), C.byref(out_r), C.byref(st))
    allow = (MEB_OK, MEB_W_NOT_CONVERGED) if allow_not_converged else (MEB_OK,)
    _check(code, "meb_solve", allow)
    return out_c, out_r.value, st.as_dict()


def meb_solve_host(ctx: Context, h_centers, h_radii, tol=1e-8, precision_mode=MEB_MODE_FP64, params=None,
                   allow_not_converged=False):
    """Same as meb_solve with HOST tensors (CPU float64, ideally pinned); H2D copies are inside the call."""
    assert (not h_centers.is_cuda) and h_centers.dtype == torch.float64 and h_centers.stride(1) == 1
    m, d = h_centers.shape
    out_c = torch.empty(d, dtype=torch.float64)
    out_r = C.c_double()
    st = meb_stats()
    code = load().meb_solve_host(ctx.h, m, d, _ptr(h_centers), h_centers.stride(0), _ptr(h_radii), float(tol),
                                 int(precision_mode), None if params is None else C.byref(params),
                                 C.c_void_p(out_c.data_ptr()), C.byref(out_r), C.byref(st))
    allow = (MEB_OK, MEB_W_NOT_CONVERGED) if allow_not_converged else (MEB_OK,)
    _check(code, "meb_solve_host", allow)
    return out_c, out_r.value, st.as_dict()


def meb_solve_sharded(ctx: Context, rank, nranks, centers_local, radii_local, row_offset, m_global, xchg_send, xchg_recv,
                      allgather, tol=1e-8, precision_mode=MEB_MODE_FP64, params=None, allow_not_converged=False):
    """This rank's rows [row_offset, row_offset + m_local) of an m_global-ball instance (CUDA float64 tensors);
    xchg_send / xchg_recv: CUDA float64 tensors of meb_shard_record_doubles(d) and nranks times that many doubles;
    allgather(n) -> 0: gathers the first n doubles of every rank's xchg_send into xchg_recv[r * n : (r + 1) * n],
    ordered on the context's stream.  Returns (center CPU tensor, radius, stats) -- identical on every rank."""
    assert centers_local.is_cuda and centers_local.dtype == torch.float64 and centers_local.stride(1) == 1
    m, d = centers_local.shape
    out_c = torch.empty(d, dtype=torch.float64)
    out_r = C.c_double()
    st = meb_stats()
    cb = ALLGATHER_FN(lambda user, n: int(allgather(int(n))))
    code = load().meb_solve_sharded(ctx.h, int(rank), int(nranks), m, int(row_offset), int(m_global), d, _ptr(centers_local),
                                    centers_local.stride(0), _ptr(radii_local), float(tol), int(precision_mode),
                                    None if params is None else C.byref(params), _ptr(xchg_send), _ptr(xchg_recv),
                                    int(xchg_send.numel()), cb, None, C.c_void_p(out_c.data_ptr()), C.byref(out_r),
                                    C.byref(st))
    allow = (MEB_OK, MEB_W_NOT_CONVERGED) if allow_not_converged else (MEB_OK,)
    _check(code, "meb_solve_sharded", allow)
    return out_c, out_r.value, st.as_dict()


def meb_shard_record_doubles(d: int) -> int:
    return int(load().meb_shard_record_doubles(int(d)))


def meb_solve_batch(ctx: Context, centers, radii, row_offsets, tol=1e-8, params=None):
    """Solves the independent small instances whose rows are row_offsets[k]:row_offsets[k+1] of `centers`
    (CUDA float64, (rows, d)) and `radii` (CUDA float64 or None) in one batch.
    Returns (centres (nprob, d) CPU tensor, radii (nprob,), status (nprob,) int32, kkt (nprob,))."""
    assert centers.is_cuda and centers.dtype == torch.float64 and centers.stride(1) == 1
    offs = torch.as_tensor(row_offsets, dtype=torch.int64).contiguous()
    nprob = offs.numel() - 1
    d = centers.shape[1]
    out_c = torch.empty((nprob, d), dtype=torch.float64)
    out_r = torch.empty(nprob, dtype=torch.float64)
    out_s = torch.empty(nprob, dtype=torch.int32)
    out_k = torch.empty(nprob, dtype=torch.float64)
    code = load().meb_solve_batch(ctx.h, nprob, C.c_void_p(offs.data_ptr()), d, _ptr(centers), centers.stride(0),
                                  _ptr(radii), float(tol), None if params is None else C.byref(params),
                                  C.c_void_p(out_c.data_ptr()), C.c_void_p(out_r.data_ptr()),
                                  C.c_void_p(out_s.data_ptr()), C.c_void_p(out_k.data_ptr()))
    _check(code, "meb_solve_batch", (MEB_OK, MEB_W_NOT_CONVERGED, MEB_E_INPUT))
    return out_c, out_r, out_s, out_k


def meb_ingest(ctx: Context, Cm, R, sample_rows=1024, want_shadow=False):
    m, d, ld, _ = _problem(MEB_FP64, Cm, R, None, None, None)
    dev = Cm.device
    c0 = torch.empty(d, dtype=torch.float64, device=dev)
    sc = torch.empty(4, dtype=torch.float64, device=dev)
    C32 = R32 = None
    ld32 = 0
    if want_shadow:
        ld32 = (d + 3) // 4 * 4
        C32 = torch.zeros((m, ld32), dtype=torch.float32, device=dev)
        R32 = torch.zeros(m, dtype=torch.float32, device=dev) if R is not None else None
    _check(load().meb_ingest(ctx.h, m, d, _ptr(Cm), ld, _ptr(R), int(sample_rows), _ptr(c0), _ptr(sc),
                             _ptr(C32), ld32, _ptr(R32)), "meb_ingest")
    s = sc.cpu()
    out = dict(c0=c0, L=float(s[0]), argmax=int(s[1]), n_bad=int(s[2]))
    if want_shadow:
        out.update(C32=C32[:, :d], R32=R32)
    return out


def meb_eval_alm(ctx: Context, prec, Cm, R, U, v_slot, Vrows, x, xbar, sigma, tau, per_ball=False,
                 active=False):
    m, d, ld, ldv = _problem(prec, Cm, R, U, v_slot, Vrows)
    dev = Cm.device
    out = torch.zeros(MEB_EVAL_NSCALARS, dtype=torch.float64, device=dev)
    grad = torch.zeros(d + 1, dtype=torch.float64, device=dev)
    t_out = torch.zeros(m, dtype=torch.float64, device=dev) if per_ball else None
    lam_out = torch.zeros(m, dtype=torch.float64, device=dev) if per_ball else None
    a_idx = torch.full((m,), -1, dtype=torch.int32, device=dev) if active else None
    a_rho = torch.zeros(m, dtype=torch.float64, device=dev) if active else None
    a_lam = torch.zeros(m, dtype=torch.float64, device=dev) if active else None
    _check(load().meb_eval_alm(ctx.h, prec, m, d, _ptr(Cm), ld, _ptr(R), _ptr(U), _ptr(v_slot), _ptr(Vrows),
                               ldv, _ptr(x), _ptr(xbar), float(sigma), float(tau), _ptr(out), _ptr(grad),
                               _ptr(t_out), _ptr(lam_out), _ptr(a_idx), _ptr(a_rho), _ptr(a_lam)),
           "meb_eval_alm")
    res = dict(scalars=out, grad=grad)
    if per_ball:
        res.update(t=t_out, lam=lam_out)
    if active:
        n = int(out[EV["N_ACTIVE"]].item())
        res.update(active_idx=a_idx[:n], active_rho=a_rho[:n], active_lam=a_lam[:n])
    return res


def meb_eval_alm_multi(ctx: Context, prec, Cm, R, U, v_slot, Vrows, x, xbar, sigma, tau, direction, gammas):
    """One pass: the evaluation at x plus psi_var at x - gammas[k] * direction (k < len(gammas) <= 4)."""
    m, d, ld, ldv = _problem(prec, Cm, R, U, v_slot, Vrows)
    dev = Cm.device
    out = torch.zeros(MEB_EVAL_NSCALARS, dtype=torch.float64, device=dev)
    grad = torch.zeros(d + 1, dtype=torch.float64, device=dev)
    n = len(gammas)
    psi = torch.zeros(n, dtype=torch.float64, device=dev)
    g = (C.c_double * n)(*[float(v) for v in gammas])
    _check(load().meb_eval_alm_multi(ctx.h, prec, m, d, _ptr(Cm), ld, _ptr(R), _ptr(U), _ptr(v_slot), _ptr(Vrows), ldv,
                                     _ptr(x), _ptr(xbar), float(sigma), float(tau), _ptr(direction), n,
                                     C.cast(g, C.c_void_p), _ptr(out), _ptr(grad), _ptr(psi)), "meb_eval_alm_multi")
    return dict(scalars=out, grad=grad, psi=psi)


def meb_hvp(ctx: Context, prec, Cm, R, U, v_slot, Vrows, x, sigma, tau, q):
    m, d, ld, ldv = _problem(prec, Cm, R, U, v_slot, Vrows)
    Hq = torch.zeros(d + 1, dtype=torch.float64, device=Cm.device)
    _check(load().meb_hvp(ctx.h, prec, m, d, _ptr(Cm), ld, _ptr(R), _ptr(U), _ptr(v_slot), _ptr(Vrows), ldv,
                          _ptr(x), float(sigma), float(tau), _ptr(q), _ptr(Hq)), "meb_hvp")
    return Hq


def meb_dense_hessian(ctx: Context, prec, Cm, R, U, v_slot, Vrows, x, sigma, tau):
    m, d, ld, ldv = _problem(prec, Cm, R, U, v_slot, Vrows)
    H = torch.zeros((d + 1, d + 1), dtype=torch.float64, device=Cm.device)
    _check(load().meb_dense_hessian(ctx.h, prec, m, d, _ptr(Cm), ld, _ptr(R), _ptr(U), _ptr(v_slot),
                                    _ptr(Vrows), ldv, _ptr(x), float(sigma), float(tau), _ptr(H)),
           "meb_dense_hessian")
    return H


def meb_update_multipliers(ctx: Context, prec, Cm, R, U, v_slot, Vrows, x, sigma, cap_rows=None):
    m, d, ld, ldv = _problem(prec, Cm, R, U, v_slot, Vrows)
    dev = Cm.device
    cap = m if cap_rows is None else int(cap_rows)
    ldo = (d + 3) // 4 * 4
    U_out = torch.empty(m, dtype=_dt(prec), device=dev)
    slot_out = torch.empty(m, dtype=torch.int32, device=dev)
    V_out = torch.zeros((max(cap, 1), ldo), dtype=_dt(prec), device=dev)
    n, s2 = C.c_int64(), C.c_double()
    code = load().meb_update_multipliers(ctx.h, prec, m, d, _ptr(Cm), ld, _ptr(R), _ptr(U), _ptr(v_slot),
                                         _ptr(Vrows), ldv, _ptr(x), float(sigma), _ptr(U_out), _ptr(slot_out),
                                         _ptr(V_out), ldo, cap, C.byref(n), C.byref(s2))
    _check(code, "meb_update_multipliers", (MEB_OK, MEB_E_CAPACITY))
    return dict(U=U_out, v_slot=slot_out, Vrows=V_out[:, :d], n_slots=n.value, sum_mult2=s2.value, code=code)


def meb_screen_compact(ctx: Context, C32, R32, r_hat, c_hat, tol_red, cap=None, flags=None,
                       flags_are_input=False):
    dev = (flags if C32 is None else C32).device
    if flags_are_input:
        m = flags.numel()
        d, ld = 1, 1
    else:
        m, d, ld, _ = _problem(MEB_FP32, C32, R32, None, None, None)
        if flags is None:
            flags = torch.zeros(m, dtype=torch.uint8, device=dev)
    cap = m if cap is None else int(cap)
    idx = torch.full((max(cap, 1),), -1, dtype=torch.int32, device=dev)
    n = C.c_int64()
    code = load().meb_screen_compact(ctx.h, m, d, _ptr(C32), ld, _ptr(R32), float(r_hat), _ptr(c_hat),
                                     float(tol_red), _ptr(idx), cap, C.byref(n), _ptr(flags),
                                     int(bool(flags_are_input)))
    _check(code, "meb_screen_compact", (MEB_OK, MEB_E_CAPACITY))
    return dict(idx=idx[:min(n.value, cap)], count=n.value, flags=flags, code=code)


def meb_feasibility_check(ctx: Context, Cm, R, r, c, eps_feas, kept_mask=None, cap=None):
    m, d, ld, _ = _problem(MEB_FP64, Cm, R, None, None, None)
    cap = m if cap is None else int(cap)
    idx = torch.full((max(cap, 1),), -1, dtype=torch.int32, device=Cm.device)
    dm, am, n = C.c_double(), C.c_int32(), C.c_int64()
    code = load().meb_feasibility_check(ctx.h, m, d, _ptr(Cm), ld, _ptr(R), float(r), _ptr(c), float(eps_feas),
                                        _ptr(kept_mask), C.byref(dm), C.byref(am), _ptr(idx), cap, C.byref(n))
    _check(code, "meb_feasibility_check", (MEB_OK, MEB_E_CAPACITY))
    return dict(delta_max=dm.value, argmax=am.value, viol_idx=idx[:min(n.value, cap)], n_viol=n.value, code=code)


MEB_STATIC_MAX_ROWS = 256 * 65536


def meb_feasibility_max_static(Cm, R, r, c, out2, stream=None):
    """Allocation-free feasibility maximum (include/meb.h a8'): the kernels are queued on ``stream`` (default: torch's
    current stream) and write (Delta_max, arg-max as a double) into the caller's device tensor ``out2``; nothing is
    allocated, copied to the host or synchronised here.  Returns the status code (MEB_E_CAPACITY beyond
    MEB_STATIC_MAX_ROWS balls).  Calls share one static device scratch: do not overlap them on the GPU."""
    m, d, ld, _ = _problem(MEB_FP64, Cm, R, None, None, None)
    assert out2.is_cuda and out2.dtype == torch.float64 and out2.is_contiguous() and out2.numel() >= 2
    assert c.is_cuda and c.dtype == torch.float64 and c.is_contiguous() and c.numel() == d
    st = torch.cuda.current_stream(Cm.device) if stream is None else stream
    code = load().meb_feasibility_max_static(C.c_void_p(st.cuda_stream), m, d, _ptr(Cm), ld, _ptr(R), float(r), _ptr(c),
                                             _ptr(out2))
    return _check(code, "meb_feasibility_max_static", (MEB_OK, MEB_E_CAPACITY))
