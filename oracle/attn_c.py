"""ctypes wrapper of oracle/echo_oracle_attn.c (the verify-attention oracle in plain C) -- TEST INFRASTRUCTURE ONLY.

Same definition and same arguments as `echo_oracle.verify_attn`; exists so that every (node, head) row of a
BASELINE.json configuration can be checked and so that the CPU baseline runs on all host cores.  Imports nothing from
the package; only tests/, __graft_entry__ and bench.py's cpu_baseline / --impl reference legs may use it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "echo_oracle_attn.c")
LIB = os.path.join(_HERE, "liboracle_attn.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math: sums run in source order), POSIX threads; rebuilt when the source is newer."""
    if force or not os.path.exists(LIB) or os.path.getmtime(SRC) > os.path.getmtime(LIB):
        cmd = [os.environ.get("CC", "gcc"), "-O2", "-std=c11", "-shared", "-fPIC", "-pthread", SRC, "-o", LIB, "-lm"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("building the C oracle failed: " + " ".join(cmd) + "\n" + r.stderr)
    return LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.oracle_verify_attn.restype = C.c_int
        lib.oracle_verify_attn.argtypes = ([C.c_void_p] * 3 + [C.c_int32] * 2 + [C.c_void_p] * 5 + [C.c_int32] * 5 +
                                           [C.c_float, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_int32])
        _lib = lib
    return _lib


def host_threads() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def verify_attn(sel, q_bits, k_pool_bits, v_pool_bits, page_table, prefix_len, Hq, Hkv, sm_scale, layer=0, rows=None,
                threads=None):
    """softmax(sm_scale q K^T) V over prefix + ancestors-or-self, fp64 (S:A-1..A-5).  Arguments as
    echo_oracle.verify_attn.  rows = None: (out [n][Hq][128], lse [n][Hq]) for all packed nodes; rows = [(k, h), ...]:
    (out [len(rows)][128], lse [len(rows)]) in that order."""
    c = lambda a, t: np.ascontiguousarray(np.asarray(a), dtype=t)
    n = int(sel["n_selected"])
    offs, req = c(sel["sel_offsets"], np.int32), c(sel["sel_req"][:n], np.int32)
    mask = c(np.asarray(sel["anc_mask"]).reshape(-1, 4)[:n], np.uint32)
    q, kp, vp = c(q_bits, np.uint16), c(k_pool_bits, np.uint16), c(v_pool_bits, np.uint16)
    pt, pl = c(page_table, np.int32), c(prefix_len, np.int32)
    assert q.ndim == 3 and q.shape[1] == Hq and q.shape[2] == 128 and q.shape[0] >= n
    assert kp.ndim == 5 and kp.shape[2] == Hkv and kp.shape[3:] == (16, 128) and kp.shape == vp.shape
    assert pt.ndim == 2 and pt.shape[0] == len(pl) == len(offs) - 1
    if rows is None:
        rr, n_rows = None, n * Hq
    else:
        rr = c(rows, np.int32).reshape(-1, 2)
        n_rows = rr.shape[0]
        assert n_rows == 0 or (0 <= rr[:, 0].min() and rr[:, 0].max() < n and 0 <= rr[:, 1].min() and rr[:, 1].max() < Hq)
    out = np.zeros((n_rows, 128), np.float64)
    lse = np.zeros(n_rows, np.float64)
    threads = host_threads() if threads is None else int(threads)
    p = lambda a: None if a is None else a.ctypes.data_as(C.c_void_p)
    rc = _load().oracle_verify_attn(p(offs), p(req), p(mask), n, len(pl), p(q), p(kp), p(vp), p(pt), p(pl), pt.shape[1],
                                    kp.shape[1], Hq, Hkv, int(layer), C.c_float(float(np.float32(sm_scale))), p(rr), n_rows,
                                    p(out), p(lse), max(1, threads))
    if rc != 0:
        raise RuntimeError("oracle_verify_attn failed (bad argument or out of memory)")
    if rows is None:
        return out.reshape(n, Hq, 128), lse.reshape(n, Hq)
    return out, lse
