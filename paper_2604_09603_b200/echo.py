"""Thin ctypes binding of libecho.so (include/echo.h).  Argument marshalling only: every step of
the hot path runs in the CUDA kernels of `csrc/`.  torch is used for device memory and streams.

There is no CPU fallback: importing works anywhere (so the symbol/ABI tests run without a GPU),
but `EchoContext()` raises unless the library loads and the device is a B200 (sm_100).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libecho.so")

ECHO_OK = 0
ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_ARCH, ERR_CUDA, ERR_TOO_LARGE = -1, -2, -3, -4, -5, -6
NOALLOC_MAX_CAND = 65536  # ECHO_NOALLOC_MAX_CAND: candidates echo_gate_select_noalloc's fixed scratch holds
OPT_FORCE_SPLITS, OPT_ATTN_PATH, OPT_NUM_CTAS, OPT_ATTN_SAFE, OPT_GATE_PATH, OPT_GATE_CLUSTER, OPT_ATTN_PLAN = 1, 2, 3, 4, 5, 6, 7
SCHED_TOPB, SCHED_ALG1 = 0, 1  # EchoGate.schedule: global top-B (north_star) / Algorithm 1 as printed
ATTN_AUTO, ATTN_SMALLROW, ATTN_TCGEN05 = 0, 1, 2
MAX_ACCEPT = 32
CUT_NEVER = 0x7FFFFFFF
DEV_BAD_PARENT, DEV_BAD_LOGQ, DEV_DEPTH_OVERFLOW, DEV_PAGE_OVERFLOW = 1, 2, 4, 8
DEV_BAD_TRACE, DEV_CALIB_OVERFLOW, DEV_TREE_OVERFLOW, DEV_CAND_OVERFLOW, DEV_INTERNAL = 16, 32, 64, 128, 256

EXPORTS = ["echo_create", "echo_destroy", "echo_workspace_bytes", "echo_strerror", "echo_last_error",
           "echo_device_status", "echo_set_option", "echo_attn_splits", "echo_launch_count", "echo_probe_sm_clock",
           "echo_gate_select", "echo_verify_attn", "echo_accept",
           "echo_calibrate", "echo_gate_keys", "echo_gate_select_keys", "echo_draft_expand",
           "echo_accept_stochastic", "echo_gate_select_noalloc", "echo_argmax_shard", "echo_argmax_merge"]


class EchoTrees(C.Structure):
    _fields_ = [("num_requests", C.c_int32), ("total_cand", C.c_int32), ("max_cand_per_req", C.c_int32),
                ("cand_offsets", C.c_void_p), ("parent", C.c_void_p), ("logq", C.c_void_p)]


class EchoGate(C.Structure):
    _fields_ = [("depth_mask", C.c_uint32), ("log_tau", C.c_float * 32), ("w_max", C.c_int32),
                ("budget", C.c_int32), ("static_k", C.c_int32), ("schedule", C.c_int32),
                ("cand_index_base", C.c_int32), ("request_base", C.c_int32)]


class EchoSelection(C.Structure):
    _fields_ = [("capacity", C.c_int32), ("n_selected", C.c_void_p), ("sel_offsets", C.c_void_p),
                ("sel_node", C.c_void_p), ("sel_req", C.c_void_p), ("parent_local", C.c_void_p),
                ("sel_depth", C.c_void_p), ("anc_mask", C.c_void_p), ("path_score", C.c_void_p),
                ("cand_depth", C.c_void_p), ("cut_depth", C.c_void_p)]


class EchoPagedKV(C.Structure):
    _fields_ = [("num_kv_heads", C.c_int32), ("head_dim", C.c_int32), ("page_size", C.c_int32),
                ("num_pages", C.c_int32), ("max_pages_per_req", C.c_int32), ("num_layers", C.c_int32),
                ("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("page_table", C.c_void_p),
                ("prefix_len", C.c_void_p)]


class EchoVerifyResult(C.Structure):
    _fields_ = [("draft_token", C.c_void_p), ("prev_token", C.c_void_p), ("target_token", C.c_void_p),
                ("target_logits", C.c_void_p), ("vocab", C.c_int32), ("ld", C.c_int64)]


class EchoAccept(C.Structure):
    _fields_ = [("accept_len", C.c_void_p), ("last_node", C.c_void_p), ("bonus_token", C.c_void_p),
                ("new_len", C.c_void_p), ("accept_idx", C.c_void_p), ("slot_src", C.c_void_p),
                ("slot_dst", C.c_void_p), ("target_token_out", C.c_void_p)]


class EchoTraces(C.Structure):
    _fields_ = [("num_samples", C.c_int64), ("depth", C.c_void_p), ("conf", C.c_void_p), ("accepted", C.c_void_p)]


class EchoCalibration(C.Structure):
    _fields_ = [("auc", C.c_void_p), ("tau", C.c_void_p), ("n_pos", C.c_void_p), ("n_neg", C.c_void_p),
                ("depth_mask", C.c_void_p)]


class EchoSampleInputs(C.Structure):
    _fields_ = [("draft_token", C.c_void_p), ("target_logits", C.c_void_p), ("root_logits", C.c_void_p),
                ("vocab", C.c_int32), ("ld", C.c_int64), ("temperature", C.c_float), ("u_accept", C.c_void_p),
                ("u_bonus", C.c_void_p)]


class EchoDraftLevel(C.Structure):
    _fields_ = [("level", C.c_int32), ("topk", C.c_int32), ("parent_score", C.c_void_p), ("child_logq", C.c_void_p),
                ("child_token", C.c_void_p)]


MAX_TOPK = 16
DEV_TREE_OVERFLOW = 64
CALIB_MAX_PER_DEPTH = 24576
CALIB_WORKSPACE_BYTES = 256 + 32 * CALIB_MAX_PER_DEPTH * 4
DEV_BAD_TRACE, DEV_CALIB_OVERFLOW = 16, 32

_lib = None


def load_library():
    """dlopen libecho.so and declare the prototypes.  Raises if the library was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2604_09603_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    P = C.POINTER
    lib.echo_create.argtypes = [P(C.c_void_p), C.c_int, C.c_size_t]
    lib.echo_create.restype = C.c_int
    lib.echo_destroy.argtypes = [C.c_void_p]
    lib.echo_destroy.restype = C.c_int
    lib.echo_workspace_bytes.argtypes = [C.c_int32] * 5
    lib.echo_attn_splits.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
    lib.echo_attn_splits.restype = C.c_int
    lib.echo_launch_count.argtypes = []
    lib.echo_launch_count.restype = C.c_uint64
    lib.echo_probe_sm_clock.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.echo_probe_sm_clock.restype = C.c_int
    lib.echo_workspace_bytes.restype = C.c_size_t
    lib.echo_strerror.argtypes = [C.c_int]
    lib.echo_strerror.restype = C.c_char_p
    lib.echo_last_error.argtypes = [C.c_void_p]
    lib.echo_last_error.restype = C.c_char_p
    lib.echo_device_status.argtypes = [C.c_void_p, P(C.c_uint32), C.c_void_p]
    lib.echo_device_status.restype = C.c_int
    lib.echo_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
    lib.echo_set_option.restype = C.c_int
    if hasattr(lib, "echo_debug_wait_prof"):  # private hook of a library built with ECHO_WAIT_PROF=1 (csrc/debug_prof.h)
        lib.echo_debug_wait_prof.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        lib.echo_debug_wait_prof.restype = C.c_int
    lib.echo_gate_keys.argtypes = [C.c_void_p, P(EchoTrees), P(EchoGate), P(EchoSelection), C.c_void_p, C.c_void_p]
    lib.echo_gate_keys.restype = C.c_int
    lib.echo_gate_select_keys.argtypes = [C.c_void_p, P(EchoTrees), P(EchoGate), C.c_void_p, C.c_void_p, C.c_int64,
                                          P(EchoSelection), C.c_void_p]
    lib.echo_gate_select_keys.restype = C.c_int
    lib.echo_accept_stochastic.argtypes = [C.c_void_p, P(EchoSelection), P(EchoSampleInputs), C.c_int32, P(EchoPagedKV),
                                           P(EchoAccept), C.c_void_p]
    lib.echo_accept_stochastic.restype = C.c_int
    lib.echo_draft_expand.argtypes = [C.c_void_p, P(EchoDraftLevel), P(EchoTrees), C.c_void_p, C.c_void_p, C.c_void_p]
    lib.echo_draft_expand.restype = C.c_int
    lib.echo_calibrate.argtypes = [C.c_void_p, P(EchoTraces), C.c_double, P(EchoCalibration), C.c_void_p]
    lib.echo_calibrate.restype = C.c_int
    lib.echo_gate_select.argtypes = [C.c_void_p, P(EchoTrees), P(EchoGate), P(EchoSelection), C.c_void_p]
    lib.echo_gate_select.restype = C.c_int
    lib.echo_gate_select_noalloc.argtypes = [P(EchoTrees), P(EchoGate), P(EchoSelection), C.c_void_p, C.c_void_p]
    lib.echo_gate_select_noalloc.restype = C.c_int
    lib.echo_verify_attn.argtypes = [C.c_void_p, P(EchoSelection), P(EchoPagedKV), C.c_int32, C.c_int32,
                                     C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p]
    lib.echo_verify_attn.restype = C.c_int
    lib.echo_argmax_shard.argtypes = [C.c_void_p, P(EchoSelection), C.c_void_p, C.c_int64, C.c_int32, C.c_int32,
                                      C.c_void_p, C.c_void_p]
    lib.echo_argmax_shard.restype = C.c_int
    lib.echo_argmax_merge.argtypes = [C.c_void_p, P(EchoSelection), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.echo_argmax_merge.restype = C.c_int
    lib.echo_accept.argtypes = [C.c_void_p, P(EchoSelection), P(EchoVerifyResult), C.c_int32, P(EchoPagedKV),
                                P(EchoAccept), C.c_void_p]
    lib.echo_accept.restype = C.c_int
    _lib = lib
    return lib


class EchoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"echo error {code}: {msg}")
        self.code = code


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


@dataclass
class Selection:
    """Device-side output of echo_gate_select (torch tensors on the context's device)."""
    capacity: int
    R: int
    n_selected: "torch.Tensor"
    sel_offsets: "torch.Tensor"
    sel_node: "torch.Tensor"
    sel_req: "torch.Tensor"
    parent_local: "torch.Tensor"
    sel_depth: "torch.Tensor"
    anc_mask: "torch.Tensor"
    path_score: "torch.Tensor"
    cand_depth: "torch.Tensor"
    cut_depth: "torch.Tensor"

    def __setattr__(self, name, value):  # a field that changes drops the marshalled struct
        self.__dict__.pop("_cs", None)
        object.__setattr__(self, name, value)

    def c_struct(self) -> EchoSelection:
        """the C struct of these tensors, marshalled once (per-call marshalling is what bounds small batches)"""
        cs = self.__dict__.get("_cs")
        if cs is None:
            cs = EchoSelection(self.capacity, _ptr(self.n_selected), _ptr(self.sel_offsets), _ptr(self.sel_node),
                               _ptr(self.sel_req), _ptr(self.parent_local), _ptr(self.sel_depth),
                               _ptr(self.anc_mask), _ptr(self.path_score), _ptr(self.cand_depth),
                               _ptr(self.cut_depth))
            self.__dict__["_cs"] = cs
        return cs

    def to_host(self) -> dict:
        """numpy copies trimmed to n_selected (synchronises)."""
        n = int(self.n_selected.item())
        return dict(n_selected=n, sel_offsets=self.sel_offsets.cpu().numpy(),
                    sel_node=self.sel_node[:n].cpu().numpy(), sel_req=self.sel_req[:n].cpu().numpy(),
                    parent_local=self.parent_local[:n].cpu().numpy(), sel_depth=self.sel_depth[:n].cpu().numpy(),
                    anc_mask=self.anc_mask[:n].cpu().numpy().view(np.uint32),
                    path_score=self.path_score.cpu().numpy(), cand_depth=self.cand_depth.cpu().numpy(),
                    cut_depth=self.cut_depth.cpu().numpy())


@dataclass
class PagedKV:
    k_pool: "torch.Tensor"      # bf16 [layers][pages][Hkv][16][128]
    v_pool: "torch.Tensor"
    page_table: "torch.Tensor"  # int32 [R][max_pages]
    prefix_len: "torch.Tensor"  # int32 [R]

    def __setattr__(self, name, value):  # a field that changes drops the marshalled structs
        self.__dict__.pop("_cs", None)
        object.__setattr__(self, name, value)

    def c_struct(self, with_pools: bool = True) -> EchoPagedKV:
        """the C struct of these tensors (pool pointers NULL if not with_pools), marshalled once"""
        cs = self.__dict__.get("_cs")
        if cs is None:
            L, NP, Hkv, PS, Dh = self.k_pool.shape
            args = (Hkv, Dh, PS, NP, self.page_table.shape[1], L)
            tail = (_ptr(self.page_table), _ptr(self.prefix_len))
            cs = (EchoPagedKV(*args, None, None, *tail), EchoPagedKV(*args, _ptr(self.k_pool), _ptr(self.v_pool), *tail))
            self.__dict__["_cs"] = cs
        return cs[1 if with_pools else 0]


@dataclass
class Acceptance:
    accept_len: "torch.Tensor"
    last_node: "torch.Tensor"
    bonus_token: "torch.Tensor"
    new_len: "torch.Tensor"
    accept_idx: "torch.Tensor"
    slot_src: "torch.Tensor"
    slot_dst: "torch.Tensor"
    target_token: Optional["torch.Tensor"]

    def __setattr__(self, name, value):  # a field that changes drops the marshalled structs
        self.__dict__.pop("_cs", None)
        object.__setattr__(self, name, value)

    def c_struct(self, with_target: bool) -> EchoAccept:
        """the C struct of these tensors (target_token_out NULL unless with_target), marshalled once"""
        cs = self.__dict__.get("_cs")
        if cs is None:
            head = (_ptr(self.accept_len), _ptr(self.last_node), _ptr(self.bonus_token), _ptr(self.new_len),
                    _ptr(self.accept_idx), _ptr(self.slot_src), _ptr(self.slot_dst))
            cs = (EchoAccept(*head, None), EchoAccept(*head, _ptr(self.target_token)))
            self.__dict__["_cs"] = cs
        return cs[1 if with_target else 0]

    def to_host(self) -> dict:
        return {k: getattr(self, k).cpu().numpy() for k in
                ("accept_len", "last_node", "bonus_token", "new_len", "accept_idx", "slot_src", "slot_dst")}


def gate_select_noalloc(cand_offsets, parent, logq, depth_mask: int, log_tau, w_max: int, budget: int, sel: "Selection",
                        status, static_k: int = 0, schedule: int = 0, max_cand: int = 128) -> "Selection":
    """echo_gate_select_noalloc: echo_gate_select without a context or workspace and without any allocation (its
    scratch is a fixed array in the library; at most NOALLOC_MAX_CAND candidates).  Runs on torch's current device
    and stream; `sel` (e.g. from EchoContext.alloc_selection) and `status` (int32 device tensor [1], flags are OR-ed
    in) are the caller's.  Calls that overlap on the GPU race on the scratch."""
    import torch
    lib = load_library()
    R, N = cand_offsets.numel() - 1, parent.numel()
    trees = EchoTrees(R, N, max_cand, _ptr(cand_offsets), _ptr(parent), _ptr(logq))
    g = EchoContext._gate_struct(depth_mask, log_tau, w_max, budget, static_k, schedule, 0, 0)
    cs = sel.c_struct()
    rc = lib.echo_gate_select_noalloc(C.byref(trees), C.byref(g), C.byref(cs), _ptr(status),
                                      C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != ECHO_OK:
        raise EchoError(rc, lib.echo_strerror(rc).decode())
    return sel


class EchoContext:
    """Owns an EchoCtx (workspace) on one CUDA device."""

    def __init__(self, device: int = 0, workspace_bytes: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("echo: no CUDA device (the hot path has no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.init()
        with torch.cuda.device(self.device):
            torch.cuda.current_stream()  # make sure the primary context exists
        self._h = C.c_void_p()
        self.workspace_bytes = int(workspace_bytes)
        rc = self.lib.echo_create(C.byref(self._h), device, self.workspace_bytes)
        if rc != ECHO_OK:
            raise EchoError(rc, self.lib.echo_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.echo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers -----------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != ECHO_OK:
            msg = self.lib.echo_strerror(rc).decode()
            if rc == ERR_CUDA:
                msg += ": " + self.lib.echo_last_error(self._h).decode()
            raise EchoError(rc, msg)

    def _stream(self):
        import torch
        return C.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    def ensure_workspace(self, R: int, N: int, capacity: int, Hq: int, Hkv: int = 0):
        key = (R, N, capacity, Hq, Hkv, self._opts.get(OPT_FORCE_SPLITS, 0) if hasattr(self, "_opts") else 0)
        if key in self.__dict__.setdefault("_ws_ok", set()):
            return
        self._ensure_workspace(R, N, capacity, Hq, Hkv)
        if len(self._ws_ok) > 1024:
            self._ws_ok.clear()
        self._ws_ok.add(key)

    def _ensure_workspace(self, R: int, N: int, capacity: int, Hq: int, Hkv: int = 0):
        splits = int(self.lib.echo_attn_splits(self._h, R, Hkv)) if Hq > 0 and Hkv > 0 else 1
        need = int(self.lib.echo_workspace_bytes(R, N, capacity, Hq, splits))
        if need > self.workspace_bytes:
            import torch
            torch.cuda.synchronize(self.device)
            opts = (self.get_options() if hasattr(self, "_opts") else {})
            self.lib.echo_destroy(self._h)
            self._h = C.c_void_p()
            self._check(self.lib.echo_create(C.byref(self._h), self.device.index, need))
            self.workspace_bytes = need
            for k, v in opts.items():
                self.set_option(k, v)

    def get_options(self) -> dict:
        return dict(getattr(self, "_opts", {}))

    def set_option(self, key: int, value: int):
        self._check(self.lib.echo_set_option(self._h, key, int(value)))
        if not hasattr(self, "_opts"):
            self._opts = {}
        self._opts[key] = int(value)

    def debug_wait_prof(self, n_ctas: int = 148):
        """[n_ctas][32] uint64 wait-cycle counters of the last tcgen05 launch (library built with ECHO_WAIT_PROF=1)."""
        import numpy as np
        if not hasattr(self.lib, "echo_debug_wait_prof"):
            raise RuntimeError("libecho.so was built without ECHO_WAIT_PROF=1")
        buf = np.zeros((n_ctas, 32), np.uint64)
        rc = self.lib.echo_debug_wait_prof(self._h, buf.ctypes.data, n_ctas)
        if rc < 0:
            self._check(rc)
        return buf[:rc]

    def launch_count(self) -> int:
        """kernels libecho.so has launched in this process so far"""
        return int(self.lib.echo_launch_count())

    def probe_sm_clock(self, out):
        """queues the SM clock probe; `out` = a float32 device tensor element (MHz, written when the stream gets there)"""
        self._check(self.lib.echo_probe_sm_clock(self._h, _ptr(out), self._stream()))

    def device_status(self) -> int:
        f = C.c_uint32(0)
        self._check(self.lib.echo_device_status(self._h, C.byref(f), self._stream()))
        return int(f.value)

    # -- the three calls ----------------------------------------------------------------------
    def alloc_selection(self, R: int, N: int, capacity: int) -> Selection:
        import torch
        d = self.device
        i32 = dict(dtype=torch.int32, device=d)
        cap = max(1, capacity)
        return Selection(capacity, R, torch.zeros(1, **i32), torch.zeros(R + 1, **i32), torch.zeros(cap, **i32),
                         torch.zeros(cap, **i32), torch.zeros(cap, **i32),
                         torch.zeros(cap, dtype=torch.uint8, device=d), torch.zeros(cap, 4, **i32),
                         torch.zeros(max(1, N), dtype=torch.float32, device=d),
                         torch.zeros(max(1, N), dtype=torch.uint8, device=d), torch.zeros(max(1, R), **i32))

    def gate_select(self, cand_offsets, parent, logq, depth_mask: int, log_tau, w_max: int, budget: int,
                    static_k: int = 0, capacity: Optional[int] = None, max_cand: int = 128,
                    out: Optional[Selection] = None, schedule: int = 0) -> Selection:
        """echo_gate_select.  cand_offsets/parent int32 and logq float32 device tensors."""
        R = cand_offsets.numel() - 1
        N = parent.numel()
        if capacity is None:
            capacity = min(N, R * static_k) if static_k > 0 else budget
        self.ensure_workspace(R, N, capacity, 0)
        sel = out if out is not None else self.alloc_selection(R, N, capacity)
        trees = EchoTrees(R, N, max_cand, _ptr(cand_offsets), _ptr(parent), _ptr(logq))
        g = self._gate_struct(depth_mask, log_tau, w_max, budget, static_k, schedule, 0, 0)
        cs = sel.c_struct()
        self._check(self.lib.echo_gate_select(self._h, C.byref(trees), C.byref(g), C.byref(cs), self._stream()))
        return sel

    _gate_cache: dict = {}

    @classmethod
    def _gate_struct(cls, depth_mask, log_tau, w_max, budget, static_k, schedule, cand_index_base, request_base):
        """EchoGate of these settings, marshalled once per distinct setting (the structs are read-only to the library)"""
        lt = np.ascontiguousarray(log_tau, np.float32)
        key = (int(depth_mask), lt.tobytes(), int(w_max), int(budget), int(static_k), int(schedule), int(cand_index_base),
               int(request_base))
        g = cls._gate_cache.get(key)
        if g is None:
            if len(cls._gate_cache) > 256:
                cls._gate_cache.clear()
            g = cls._gate_cache[key] = cls._make_gate_struct(*key[:1], lt, *key[2:])
        return g

    @staticmethod
    def _make_gate_struct(depth_mask, log_tau, w_max, budget, static_k, schedule, cand_index_base, request_base):
        g = EchoGate()
        g.depth_mask = int(depth_mask) & 0xFFFFFFFF
        lt = np.asarray(log_tau, np.float32)
        for d in range(32):
            g.log_tau[d] = float(lt[d])
        g.w_max, g.budget, g.static_k, g.schedule = int(w_max), int(budget), int(static_k), int(schedule)
        g.cand_index_base, g.request_base = int(cand_index_base), int(request_base)
        return g

    def gate_keys(self, cand_offsets, parent, logq, depth_mask: int, log_tau, w_max: int, budget: int, sel: Selection,
                  static_k: int = 0, schedule: int = 0, cand_index_base: int = 0, request_base: int = 0,
                  max_cand: int = 128):
        """echo_gate_keys: S1-S2 and the selection keys of this rank's candidates -> int64 device tensor [N]
        (the bits of the uint64 keys; -1 = not eligible), to be all-gathered across the ranks sharing the budget.
        The tensor is a buffer this context reuses on the next call."""
        import torch
        R, N = cand_offsets.numel() - 1, parent.numel()
        if getattr(self, "_keys_buf", None) is None or self._keys_buf.numel() < max(1, N):
            self._keys_buf = torch.empty(max(1, N), dtype=torch.int64, device=self.device)
        keys = self._keys_buf
        trees = EchoTrees(R, N, max_cand, _ptr(cand_offsets), _ptr(parent), _ptr(logq))
        g = self._gate_struct(depth_mask, log_tau, w_max, budget, static_k, schedule, cand_index_base, request_base)
        cs = sel.c_struct()
        self._check(self.lib.echo_gate_keys(self._h, C.byref(trees), C.byref(g), C.byref(cs), _ptr(keys), self._stream()))
        return keys[:N]

    def gate_select_keys(self, cand_offsets, parent, logq, depth_mask: int, log_tau, w_max: int, budget: int,
                         local_keys, all_keys, sel: Selection, static_k: int = 0, schedule: int = 0,
                         max_cand: int = 128) -> Selection:
        """echo_gate_select_keys: threshold over `all_keys` (every rank's keys), packing of this rank's requests."""
        R, N = cand_offsets.numel() - 1, parent.numel()
        self.ensure_workspace(R, N, sel.capacity, 0)
        trees = EchoTrees(R, N, max_cand, _ptr(cand_offsets), _ptr(parent), _ptr(logq))
        g = self._gate_struct(depth_mask, log_tau, w_max, budget, static_k, schedule, 0, 0)
        cs = sel.c_struct()
        self._check(self.lib.echo_gate_select_keys(self._h, C.byref(trees), C.byref(g), _ptr(local_keys), _ptr(all_keys),
                                                   int(all_keys.numel()), C.byref(cs), self._stream()))
        return sel

    def verify_attn(self, sel: Selection, kv: PagedKV, q, sm_scale: float, layer: int = 0, out=None, lse=None):
        """echo_verify_attn.  q bf16 [capacity][Hq][128] -> (out bf16 same shape, lse f32 [capacity][Hq])."""
        import torch
        Hq = q.shape[1]
        self.ensure_workspace(sel.R, 0, sel.capacity, Hq, kv.k_pool.shape[2])
        if out is None:
            out = torch.zeros_like(q)
        if lse is None:
            lse = torch.zeros(q.shape[0], Hq, dtype=torch.float32, device=q.device)
        cs, ck = sel.c_struct(), kv.c_struct()
        self._check(self.lib.echo_verify_attn(self._h, C.byref(cs), C.byref(ck), layer, Hq, sel.R, _ptr(q),
                                              _ptr(out), _ptr(lse), C.c_float(sm_scale), self._stream()))
        return out, lse

    def alloc_accept(self, R: int, capacity: int) -> Acceptance:
        import torch
        i32 = dict(dtype=torch.int32, device=self.device)
        r = max(1, R)
        return Acceptance(torch.zeros(r, **i32), torch.zeros(r, **i32), torch.zeros(r, **i32),
                          torch.zeros(r, **i32), torch.zeros(r, MAX_ACCEPT, **i32),
                          torch.zeros(r, MAX_ACCEPT, **i32), torch.zeros(r, MAX_ACCEPT, **i32),
                          torch.zeros(max(1, capacity), **i32))

    def accept_stochastic(self, sel: Selection, kv: PagedKV, draft_token, target_logits, root_logits, vocab: int,
                          temperature: float, u_accept, u_bonus, out: Optional[Acceptance] = None,
                          compact: bool = True) -> Acceptance:
        """echo_accept_stochastic.  target_logits bf16 [capacity][ld], root_logits bf16 [R][ld] (same pitch),
        u_accept f32 [capacity], u_bonus f32 [R]."""
        acc = out if out is not None else self.alloc_accept(sel.R, sel.capacity)
        self.ensure_workspace(sel.R, 0, sel.capacity, 0)
        assert target_logits.stride(0) == root_logits.stride(0)
        inp = EchoSampleInputs(_ptr(draft_token), _ptr(target_logits), _ptr(root_logits), int(vocab),
                               int(root_logits.stride(0)), float(temperature), _ptr(u_accept), _ptr(u_bonus))
        ck = kv.c_struct(with_pools=compact)
        oa = acc.c_struct(with_target=False)
        cs = sel.c_struct()
        self._check(self.lib.echo_accept_stochastic(self._h, C.byref(cs), C.byref(inp), sel.R, C.byref(ck), C.byref(oa),
                                                    self._stream()))
        return acc

    def draft_expand(self, level: int, topk: int, parent_score, child_logq, child_token, cand_offsets, parent, logq,
                     token, score_out, max_cand: int = 128):
        """echo_draft_expand: appends level `level` (topk nodes per request) to the candidate trees in place.
        parent_score f32 [R][k_prev], child_logq f32 / child_token i32 [R][k_prev][topk]; cand_offsets / parent / logq
        are the EchoTrees arrays, token i32 [N], score_out f32 [R][topk] (the next level's parent_score)."""
        R = cand_offsets.numel() - 1
        lv = EchoDraftLevel(int(level), int(topk), _ptr(parent_score), _ptr(child_logq), _ptr(child_token))
        trees = EchoTrees(R, parent.numel(), max_cand, _ptr(cand_offsets), _ptr(parent), _ptr(logq))
        self._check(self.lib.echo_draft_expand(self._h, C.byref(lv), C.byref(trees), _ptr(token), _ptr(score_out),
                                               self._stream()))
        return score_out

    def calibrate(self, depth, conf, accepted, delta: float):
        """echo_calibrate.  depth / accepted uint8 and conf float32 device tensors of M warm-up samples ->
        dict of device tensors auc f64[32], tau f32[32], n_pos / n_neg i32[32], depth_mask i32[1] (bits)."""
        import torch
        if self.workspace_bytes < CALIB_WORKSPACE_BYTES:
            torch.cuda.synchronize(self.device)
            opts = self.get_options()
            self.lib.echo_destroy(self._h)
            self._h = C.c_void_p()
            self._check(self.lib.echo_create(C.byref(self._h), self.device.index, CALIB_WORKSPACE_BYTES))
            self.workspace_bytes = CALIB_WORKSPACE_BYTES
            for k_, v_ in opts.items():
                self.set_option(k_, v_)
        d = self.device
        out = dict(auc=torch.zeros(32, dtype=torch.float64, device=d), tau=torch.zeros(32, dtype=torch.float32, device=d),
                   n_pos=torch.zeros(32, dtype=torch.int32, device=d), n_neg=torch.zeros(32, dtype=torch.int32, device=d),
                   depth_mask=torch.zeros(1, dtype=torch.int32, device=d))
        tr = EchoTraces(int(conf.numel()), _ptr(depth), _ptr(conf), _ptr(accepted))
        oc = EchoCalibration(_ptr(out["auc"]), _ptr(out["tau"]), _ptr(out["n_pos"]), _ptr(out["n_neg"]),
                             _ptr(out["depth_mask"]))
        self._check(self.lib.echo_calibrate(self._h, C.byref(tr), C.c_double(delta), C.byref(oc), self._stream()))
        return out

    def argmax_shard(self, sel: Selection, logits_shard, vocab_base: int, vocab_shard: Optional[int] = None, out=None):
        """echo_argmax_shard: logits_shard bf16 [capacity][ld], this rank's columns [vocab_base, vocab_base +
        vocab_shard) of the target logits -> int64 [capacity] (max, first index) keys to all-gather."""
        import torch
        if out is None:
            out = torch.empty(max(1, sel.capacity), dtype=torch.int64, device=self.device)
        n = int(logits_shard.shape[1] if vocab_shard is None else vocab_shard)
        cs = sel.c_struct()
        self._check(self.lib.echo_argmax_shard(self._h, C.byref(cs), _ptr(logits_shard), int(logits_shard.stride(0)), n,
                                               int(vocab_base), _ptr(out), self._stream()))
        return out

    def argmax_merge(self, sel: Selection, pairs_all, world: int, out=None):
        """echo_argmax_merge: pairs_all int64 [world][capacity] (the ranks' gathered keys) -> int32 [capacity] target
        tokens (rows < n_selected), to be passed to accept(target_token=...)."""
        import torch
        if out is None:
            out = torch.zeros(max(1, sel.capacity), dtype=torch.int32, device=self.device)
        cs = sel.c_struct()
        self._check(self.lib.echo_argmax_merge(self._h, C.byref(cs), _ptr(pairs_all), int(world), _ptr(out),
                                               self._stream()))
        return out

    def accept(self, sel: Selection, kv: PagedKV, draft_token, prev_token, target_token=None,
               target_logits=None, vocab: int = 0, out: Optional[Acceptance] = None,
               compact: bool = True) -> Acceptance:
        """echo_accept.  Exactly one of target_token (int32 [capacity]) / target_logits (bf16 [capacity][ld])."""
        acc = out if out is not None else self.alloc_accept(sel.R, sel.capacity)
        self.ensure_workspace(sel.R, 0, sel.capacity, 0)
        res = EchoVerifyResult(_ptr(draft_token), _ptr(prev_token), _ptr(target_token), _ptr(target_logits),
                               int(vocab), int(target_logits.stride(0)) if target_logits is not None else 0)
        ck = kv.c_struct(with_pools=compact)
        oa = acc.c_struct(with_target=target_logits is not None)
        cs = sel.c_struct()
        self._check(self.lib.echo_accept(self._h, C.byref(cs), C.byref(res), sel.R, C.byref(ck), C.byref(oa),
                                         self._stream()))
        return acc
