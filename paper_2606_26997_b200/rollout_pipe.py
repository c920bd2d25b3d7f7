"""ctypes binding of include/rollout_pipe.h (host-side RolloutPipe scheduler model).
Argument marshalling only; the model runs in csrc/rollout_pipe.cpp inside libgrpo_b200.so."""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from .binding import load_library

RP_EXPORTS = ["rp_fgd_frontier", "rp_rollout", "rp_cgp_timeline", "rp_simulate"]
MODE_SLIME, MODE_CGP, MODE_CGP_FGD = 0, 1, 2


class RpTimeline(C.Structure):
    _fields_ = [("t_first_U", C.c_double), ("t_complete", C.c_double), ("dt_cgp", C.c_double),
                ("t_start", C.c_double), ("t_train_end", C.c_double), ("compute", C.c_double), ("wait", C.c_double),
                ("w_train_eq4", C.c_double), ("w_train_alt", C.c_double), ("n_updates", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_READY = False


def _lib():
    global _READY
    lib = load_library()
    if not _READY:
        vp, i32, f64 = C.c_void_p, C.c_int32, C.c_double
        for name in RP_EXPORTS:
            getattr(lib, name).restype = i32
        lib.rp_fgd_frontier.argtypes = [vp, i32, i32, vp, C.POINTER(i32)]
        lib.rp_rollout.argtypes = [vp, i32, i32, f64, f64, i32, vp, vp, vp, vp, i32, C.POINTER(i32)]
        lib.rp_cgp_timeline.argtypes = [vp, vp, i32, i32, i32, C.POINTER(RpTimeline), vp, vp, vp, vp]
        lib.rp_simulate.argtypes = [vp, i32, i32, f64, f64, i32, i32, i32, vp, vp, C.POINTER(RpTimeline), vp, vp, vp,
                                    vp, vp]
        _READY = True
    return lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _ok(st: int, what: str):
    if st != 0:
        raise ValueError(f"{what}: status {st} (bad argument)")


def rp_fgd_frontier(orders: Sequence[int], F_w: int):
    o = np.ascontiguousarray(np.asarray(orders, dtype=np.int64))
    out = np.empty(max(min(F_w, o.size), 0), dtype=np.int64)
    n = C.c_int32(0)
    _ok(_lib().rp_fgd_frontier(_p(o), o.size, F_w, _p(out), C.byref(n)), "rp_fgd_frontier")
    return out[:n.value].tolist()


def rp_rollout(work, capacity: float, max_rate: float = 0.0, F_w: int = 0, trace_cap: int = 0):
    w = _f64(work)
    R, K = w.shape
    rd, gd = np.empty((R, K)), np.empty(R)
    tt = np.empty(max(trace_cap, 1))
    tg = np.full((max(trace_cap, 1), max(F_w, 1)), -1, dtype=np.int64)
    n = C.c_int32(0)
    _ok(_lib().rp_rollout(_p(w), R, K, capacity, max_rate, F_w, _p(rd), _p(gd), _p(tt), _p(tg), trace_cap,
                          C.byref(n)), "rp_rollout")
    k = min(n.value, trace_cap)
    trace = [(float(tt[i]), [int(g) for g in tg[i] if g >= 0]) for i in range(k)]
    return rd, gd, trace


def rp_cgp_timeline(trainable, train_s, U: int, mode: int):
    tr, ts = _f64(trainable), _f64(train_s)
    R = tr.size
    n_upd = (R + U - 1) // max(U, 1)
    out = RpTimeline()
    fifo = np.empty(R, dtype=np.int32)
    ready, start, end = np.empty(n_upd), np.empty(n_upd), np.empty(n_upd)
    _ok(_lib().rp_cgp_timeline(_p(tr), _p(ts), R, U, mode, C.byref(out), _p(fifo), _p(ready), _p(start), _p(end)),
        "rp_cgp_timeline")
    d = out.as_dict()
    d.update(fifo_order=fifo.tolist(), ready=ready.tolist(), start=start.tolist(), end=end.tolist())
    return d


def rp_simulate(work, capacity: float, max_rate: float, F_w: int, U: int, mode: int, materialize_s, train_s):
    w, ms, ts = _f64(work), _f64(materialize_s), _f64(train_s)
    R, K = w.shape
    n_upd = (R + U - 1) // max(U, 1)
    out = RpTimeline()
    trn = np.empty(R)
    fifo = np.empty(R, dtype=np.int32)
    ready, start, end = np.empty(n_upd), np.empty(n_upd), np.empty(n_upd)
    _ok(_lib().rp_simulate(_p(w), R, K, capacity, max_rate, F_w, U, mode, _p(ms), _p(ts), C.byref(out), _p(trn),
                           _p(fifo), _p(ready), _p(start), _p(end)), "rp_simulate")
    d = out.as_dict()
    d.update(trainable=trn, fifo_order=fifo.tolist(), ready=ready.tolist(), start=start.tolist(), end=end.tolist())
    return d
