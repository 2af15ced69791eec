"""Thin Python binding of the C-ABI library (include/foremoe.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libforemoe.so``; PyTorch supplies device
memory and streams.  There is no CPU fallback: importing the library fails loudly when the
extension has not been built (``python -m paper_2606_11867_b200.build``).

Function names and arguments mirror the header: ``load_hist``, ``assign``, ``dispatch``,
``combine``, ``workspace_bytes``, ``step_host``.  Tensors must be contiguous; device entry points
take CUDA tensors and enqueue on the current stream without synchronising.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
from typing import Optional

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libforemoe.so")

OK = 0
ERR_INVALID_ARG = -1
ERR_WORKSPACE = -2
ERR_CUDA = -3

FAULT_ID_RANGE = 1
FAULT_NO_HOST = 2
FAULT_SLOT_EXPERT = 4
FAULT_MB_OFF = 8
FAULT_QUOTA_IN = 16
FAULT_SOURCE = 32

ACT_BF16 = 0
ACT_FP32 = 1

FLAG_PLAN_STABLE = 1

EXPORTS = ("foremoe_version", "foremoe_workspace_bytes", "foremoe_warmup", "foremoe_load_hist", "foremoe_assign",
           "foremoe_plan", "foremoe_plan_noalloc",
           "foremoe_dispatch", "foremoe_combine", "foremoe_combine_bwd", "foremoe_dispatch_bwd",
           "foremoe_base_placement", "foremoe_base_placement_machines", "foremoe_source_ids", "foremoe_local_placement", "foremoe_traffic",
           "foremoe_local_placement_theta", "foremoe_tradeoff_select",
           "foremoe_swap_relocation", "foremoe_replication", "foremoe_replica_search",
           "foremoe_microstep_placement", "foremoe_step_host_arena_bytes", "foremoe_step_host")


class ForeMoEError(RuntimeError):
    def __init__(self, fn: str, code: int):
        names = {ERR_INVALID_ARG: "INVALID_ARG", ERR_WORKSPACE: "WORKSPACE_TOO_SMALL",
                 ERR_CUDA: "CUDA_ERROR"}
        super().__init__(f"{fn} failed: {names.get(code, code)}")
        self.code = code


class _CShape(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("L", "E", "K", "P", "Nb", "Nr", "T", "n_mb", "H",
                                         "act_dtype", "placement_mb_stride", "flags")]


@dataclasses.dataclass
class Shape:
    """foremoe_shape_t (Table 1 notation)."""
    L: int
    E: int
    K: int
    P: int
    Nb: int
    Nr: int
    T: int
    n_mb: int
    H: int
    act_dtype: int = ACT_BF16
    placement_mb_stride: int = 0
    flags: int = 0              # FLAG_PLAN_STABLE: see include/foremoe.h, "Stream order"

    @property
    def Ns(self) -> int:
        return self.Nb + self.Nr

    @property
    def S(self) -> int:
        return self.P * self.Ns

    @property
    def act_torch_dtype(self):
        return torch.bfloat16 if self.act_dtype == ACT_BF16 else torch.float32

    def c(self) -> _CShape:
        """The C struct (cached per field tuple: the per-instance calls of a step reuse it)."""
        key = (self.L, self.E, self.K, self.P, self.Nb, self.Nr, self.T, self.n_mb, self.H,
               self.act_dtype, self.placement_mb_stride, self.flags)
        hit = _shape_cache.get(key)
        if hit is None:
            if len(_shape_cache) > 256:
                _shape_cache.clear()
            hit = _shape_cache[key] = _CShape(*key)
        return hit


_shape_cache: dict = {}


_lib = None


def lib() -> C.CDLL:
    """The loaded C-ABI library.  Raises if it was not built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2606_11867_b200.build` "
                "(the ForeMoE path has no CPU or PyTorch fallback)")
        l = C.CDLL(LIB_PATH)
        vp, i32, sz = C.c_void_p, C.c_int32, C.c_size_t
        sp = C.POINTER(_CShape)
        l.foremoe_version.restype = C.c_int
        l.foremoe_version.argtypes = []
        l.foremoe_workspace_bytes.argtypes = [sp, C.POINTER(sz)]
        l.foremoe_warmup.argtypes = [sp, vp]
        l.foremoe_load_hist.argtypes = [sp, vp, vp, vp, vp, vp, vp]
        l.foremoe_assign.argtypes = [sp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp]
        l.foremoe_plan.argtypes = [sp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp]
        l.foremoe_plan_noalloc.argtypes = [sp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_dispatch.argtypes = [sp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_combine.argtypes = [sp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_combine_bwd.argtypes = [sp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_dispatch_bwd.argtypes = [sp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
        l.foremoe_base_placement.argtypes = [sp, vp, vp, vp, vp]
        l.foremoe_base_placement_machines.argtypes = [sp, i32, C.c_int64, C.c_int64, vp, vp, vp, vp]
        l.foremoe_source_ids.argtypes = [sp, i32, vp, vp, vp, vp, vp]
        l.foremoe_local_placement.argtypes = [sp, i32, vp, vp, vp, vp]
        l.foremoe_traffic.argtypes = [sp, i32, vp, vp, vp]
        l.foremoe_local_placement_theta.argtypes = [sp, i32, C.c_int64, C.c_int64, vp, vp, vp, vp, vp]
        l.foremoe_tradeoff_select.argtypes = [sp, i32, i32, C.c_int64, C.c_int64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_replication.argtypes = [sp, i32, vp, vp, vp, vp, vp]
        l.foremoe_replica_search.argtypes = [sp, i32, i32, C.c_int64, C.c_int64, vp, vp, vp, vp, vp, vp, vp]
        l.foremoe_swap_relocation.argtypes = [sp, i32, i32, i32, C.c_int64, C.c_int64, vp, vp, vp, vp, vp, vp]
        l.foremoe_microstep_placement.argtypes = [sp, i32, vp, vp, vp, vp, vp]
        l.foremoe_step_host_arena_bytes.argtypes = [sp, vp, C.POINTER(sz)]
        l.foremoe_step_host.argtypes = [sp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp]
        for name in EXPORTS:
            getattr(l, name).restype = C.c_int
        _lib = l
    return _lib


def _dev(t: Optional[torch.Tensor], dtype=None) -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if not t.is_contiguous():
        raise ValueError("expected a contiguous tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


def _host(t: Optional[torch.Tensor], dtype=None) -> Optional[int]:
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous host tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


_raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)


def _stream() -> int:
    """cudaStream_t of torch's current stream on the current device (the raw getter avoids building a
    Stream object per call: the per-instance calls of small micro-steps are host-bound)."""
    if _raw_stream is not None:
        return _raw_stream(torch.cuda.current_device())
    return torch.cuda.current_stream().cuda_stream


def _stream_on(dev_index: int) -> int:
    """cudaStream_t of torch's current stream on device ``dev_index`` (DataPath: the plan's device);
    falls back to the public API when the torch build lacks the raw getter, like ``_stream``."""
    if _raw_stream is not None:
        return _raw_stream(dev_index)
    return torch.cuda.current_stream(dev_index).cuda_stream


def _check(fn: str, rc: int) -> None:
    if rc != OK:
        raise ForeMoEError(fn, rc)


def version() -> int:
    return lib().foremoe_version()


def workspace_bytes(shape: Shape) -> int:
    out = C.c_size_t(0)
    _check("foremoe_workspace_bytes", lib().foremoe_workspace_bytes(C.byref(shape.c()), C.byref(out)))
    return out.value


def warmup(shape: Shape) -> None:
    """Prepare every data-path kernel variant of this shape on the current device (no launch): after
    it the data-path calls can be captured into a CUDA graph from the first call on."""
    _check("foremoe_warmup", lib().foremoe_warmup(C.byref(shape.c()), _stream()))


def load_hist(shape: Shape, ids, mb_off, hist, step_hist=None, dev_status=None) -> None:
    """(a1) hist[n_mb,L,E] int32 (and step_hist[L,E] int64) from ids[L,T,K], mb_off[n_mb+1]."""
    _check("foremoe_load_hist", lib().foremoe_load_hist(
        C.byref(shape.c()), _dev(ids, torch.int32), _dev(mb_off, torch.int32),
        _dev(hist, torch.int32), _dev(step_hist, torch.int64), _dev(dev_status, torch.int32),
        _stream()))


def assign(shape: Shape, ids, mb_off, hist, slot_expert, quota_in, quota, rank_load, slot_off,
           pair_slot, inv, workspace, dev_status=None) -> None:
    """(a2-a4) quotas, rank loads, slot offsets, pair_slot and inv for every instance."""
    _check("foremoe_assign", lib().foremoe_assign(
        C.byref(shape.c()), _dev(ids, torch.int32), _dev(mb_off, torch.int32),
        _dev(hist, torch.int32), _dev(slot_expert, torch.int32), _dev(quota_in, torch.int32),
        _dev(quota, torch.int32), _dev(rank_load, torch.int32), _dev(slot_off, torch.int32),
        _dev(pair_slot, torch.int32), _dev(inv, torch.int32), _dev(workspace),
        workspace.numel() * workspace.element_size(), _dev(dev_status, torch.int32), _stream()))


def plan(shape: Shape, ids, mb_off, slot_expert, quota_in, hist, step_hist, quota, rank_load, slot_off,
         pair_slot, inv, workspace, dev_status=None) -> None:
    """(a1-a4) load_hist + assign in two passes over the ids; hist / step_hist are outputs."""
    _check("foremoe_plan", lib().foremoe_plan(
        C.byref(shape.c()), _dev(ids, torch.int32), _dev(mb_off, torch.int32),
        _dev(slot_expert, torch.int32), _dev(quota_in, torch.int32), _dev(hist, torch.int32),
        _dev(step_hist, torch.int64), _dev(quota, torch.int32), _dev(rank_load, torch.int32),
        _dev(slot_off, torch.int32), _dev(pair_slot, torch.int32), _dev(inv, torch.int32), _dev(workspace),
        workspace.numel() * workspace.element_size(), _dev(dev_status, torch.int32), _stream()))


NOALLOC_SCRATCH_BYTES = 8 << 20     # FOREMOE_NOALLOC_SCRATCH_BYTES of include/foremoe.h


def plan_noalloc(shape: Shape, ids, mb_off, slot_expert, quota_in, hist, step_hist, quota, rank_load,
                 slot_off, pair_slot, inv, dev_status=None) -> None:
    """``plan`` without a workspace argument, for callers that cannot allocate device memory where they
    plan (a guest of an engine that reserved all of HBM, a host that forbids allocation after start-up,
    a loop that must not take cudaMalloc's device-wide sync).  The scratch is an 8 MiB array built into
    the library, one per GPU, shared by every call: shapes whose ``workspace_bytes`` exceed
    ``NOALLOC_SCRATCH_BYTES`` are refused, and calls that could overlap on the GPU (two streams, no
    event between them) corrupt each other -- keep them on one stream or order them.  Make the first
    call on a device an eager one (it looks the array's address up).  Outputs equal ``plan``'s."""
    need = workspace_bytes(shape)
    if need > NOALLOC_SCRATCH_BYTES:        # same refusal as the C entry point's, with both numbers spelled out
        err = ForeMoEError("foremoe_plan_noalloc", ERR_WORKSPACE)
        err.args = (f"foremoe_plan_noalloc: this shape needs {need} bytes of scratch, the built-in array holds "
                    f"{NOALLOC_SCRATCH_BYTES}; use plan() with a caller-owned workspace",)
        raise err
    _check("foremoe_plan_noalloc", lib().foremoe_plan_noalloc(
        C.byref(shape.c()), _dev(ids, torch.int32), _dev(mb_off, torch.int32),
        _dev(slot_expert, torch.int32), _dev(quota_in, torch.int32), _dev(hist, torch.int32),
        _dev(step_hist, torch.int64), _dev(quota, torch.int32), _dev(rank_load, torch.int32),
        _dev(slot_off, torch.int32), _dev(pair_slot, torch.int32), _dev(inv, torch.int32),
        _dev(dev_status, torch.int32), _stream()))


def dispatch(shape: Shape, layer: int, mb_begin: int, mb_end: int, mb_off, inv, x, perm, buf,
             dev_status=None) -> None:
    """(a4-a5) perm[T_range*K] and buf[T_range*K,H] for micro-steps [mb_begin, mb_end)."""
    _check("foremoe_dispatch", lib().foremoe_dispatch(
        C.byref(shape.c()), layer, mb_begin, mb_end, _dev(mb_off, torch.int32),
        _dev(inv, torch.int32), _dev(x, shape.act_torch_dtype), _dev(perm, torch.int32),
        _dev(buf, shape.act_torch_dtype), _dev(dev_status, torch.int32), _stream()))


def combine(shape: Shape, layer: int, mb_begin: int, mb_end: int, mb_off, inv, w, expert_out, y,
            dev_status=None) -> None:
    """(a6) y[T_range,H] fp32 = weighted top-K sum of expert_out rows."""
    _check("foremoe_combine", lib().foremoe_combine(
        C.byref(shape.c()), layer, mb_begin, mb_end, _dev(mb_off, torch.int32),
        _dev(inv, torch.int32), _dev(w, torch.float32), _dev(expert_out, shape.act_torch_dtype),
        _dev(y, torch.float32), _dev(dev_status, torch.int32), _stream()))


def combine_bwd(shape: Shape, layer: int, mb_begin: int, mb_end: int, mb_off, inv, w, dy, expert_out,
                d_expert_out, dw=None, dev_status=None) -> None:
    """(f.3) d_expert_out[T_range*K,H] = w * dy scattered to slot order; dw[L,T,K] = <dy, expert_out>."""
    _check("foremoe_combine_bwd", lib().foremoe_combine_bwd(
        C.byref(shape.c()), layer, mb_begin, mb_end, _dev(mb_off, torch.int32),
        _dev(inv, torch.int32), _dev(w, torch.float32), _dev(dy, torch.float32),
        _dev(expert_out, shape.act_torch_dtype), _dev(d_expert_out, shape.act_torch_dtype),
        _dev(dw, torch.float32), _dev(dev_status, torch.int32), _stream()))


def dispatch_bwd(shape: Shape, layer: int, mb_begin: int, mb_end: int, mb_off, inv, d_buf, dx,
                 dev_status=None) -> None:
    """(f.3) dx[T_range,H] fp32 = sum of the K gradient rows of every token."""
    _check("foremoe_dispatch_bwd", lib().foremoe_dispatch_bwd(
        C.byref(shape.c()), layer, mb_begin, mb_end, _dev(mb_off, torch.int32),
        _dev(inv, torch.int32), _dev(d_buf, shape.act_torch_dtype), _dev(dx, torch.float32),
        _dev(dev_status, torch.int32), _stream()))


class DataPath:
    """The data-path calls of ONE plan with the plan's own arguments marshalled once.

    The per-instance calls of small micro-steps are host-bound (about 7 us of argument checking and
    ctypes conversion per call through the functions above, against 10-20 us of kernel time for a
    one-sample micro-step): this object validates shape, mb_off, inv, w and dev_status when it is
    built and keeps their C forms, so that a call converts only the activations it is given.  Same
    C entry points, same semantics; the tensors must stay alive and unmoved while it is used."""

    def __init__(self, shape: Shape, mb_off, inv, w, dev_status=None):
        self.shape = shape
        self._keep = (mb_off, inv, w, dev_status)
        self._sp = C.byref(shape.c())
        self._mb = C.c_void_p(_dev(mb_off, torch.int32))
        self._inv = C.c_void_p(_dev(inv, torch.int32))
        self._w = C.c_void_p(_dev(w, torch.float32))
        self._st = C.c_void_p(_dev(dev_status, torch.int32))
        self._act = shape.act_torch_dtype
        l = lib()
        self._dispatch, self._combine = l.foremoe_dispatch, l.foremoe_combine
        self._combine_bwd, self._dispatch_bwd = l.foremoe_combine_bwd, l.foremoe_dispatch_bwd
        self._dev_index = inv.device.index

    def _act_ptr(self, t) -> int:
        if t.dtype != self._act or not t.is_cuda or not t.is_contiguous():
            raise ValueError(f"expected a contiguous CUDA tensor of dtype {self._act}")
        return t.data_ptr()

    @staticmethod
    def _f32_ptr(t) -> int:
        if t.dtype != torch.float32 or not t.is_cuda or not t.is_contiguous():
            raise ValueError("expected a contiguous CUDA float32 tensor")
        return t.data_ptr()

    def dispatch(self, layer: int, mb_begin: int, mb_end: int, x, perm, buf) -> None:
        rc = self._dispatch(self._sp, layer, mb_begin, mb_end, self._mb, self._inv, self._act_ptr(x),
                            None if perm is None else _dev(perm, torch.int32), self._act_ptr(buf), self._st,
                            _stream_on(self._dev_index))
        if rc:
            raise ForeMoEError("foremoe_dispatch", rc)

    def combine(self, layer: int, mb_begin: int, mb_end: int, expert_out, y) -> None:
        rc = self._combine(self._sp, layer, mb_begin, mb_end, self._mb, self._inv, self._w,
                           self._act_ptr(expert_out), self._f32_ptr(y), self._st, _stream_on(self._dev_index))
        if rc:
            raise ForeMoEError("foremoe_combine", rc)

    def combine_bwd(self, layer: int, mb_begin: int, mb_end: int, dy, expert_out, d_expert_out, dw=None) -> None:
        rc = self._combine_bwd(self._sp, layer, mb_begin, mb_end, self._mb, self._inv, self._w,
                               self._f32_ptr(dy), None if expert_out is None else self._act_ptr(expert_out),
                               self._act_ptr(d_expert_out), None if dw is None else self._f32_ptr(dw),
                               self._st, _stream_on(self._dev_index))
        if rc:
            raise ForeMoEError("foremoe_combine_bwd", rc)

    def dispatch_bwd(self, layer: int, mb_begin: int, mb_end: int, d_buf, dx) -> None:
        rc = self._dispatch_bwd(self._sp, layer, mb_begin, mb_end, self._mb, self._inv, self._act_ptr(d_buf),
                                self._f32_ptr(dx), self._st, _stream_on(self._dev_index))
        if rc:
            raise ForeMoEError("foremoe_dispatch_bwd", rc)


def base_placement(shape: Shape, step_hist, slot_expert, dev_status=None) -> None:
    """(f.4) Stage-1 rank-level LPT: step_hist int64 [L,E] -> slot_expert int32 [L,S]."""
    _check("foremoe_base_placement", lib().foremoe_base_placement(
        C.byref(shape.c()), _dev(step_hist, torch.int64), _dev(slot_expert, torch.int32),
        _dev(dev_status, torch.int32), _stream()))


def base_placement_machines(shape: Shape, M: int, a: int, b: int, step_hist_v, slot_expert,
                            dev_status=None) -> None:
    """(f.4) Alg. 1 in full: step_hist_v int64 [L,E*M] -> slot_expert int32 [L,S]."""
    _check("foremoe_base_placement_machines", lib().foremoe_base_placement_machines(
        C.byref(shape.c()), M, a, b, _dev(step_hist_v, torch.int64), _dev(slot_expert, torch.int32),
        _dev(dev_status, torch.int32), _stream()))


def microstep_placement(shape: Shape, M: int, hist, base_slot_expert, slot_expert_mb,
                        dev_status=None) -> None:
    """(f.2) Alg. 3 Stages 2-3: hist [n_mb,L,E] + base [L,S] -> slot_expert_mb [n_mb,L,S]."""
    _check("foremoe_microstep_placement", lib().foremoe_microstep_placement(
        C.byref(shape.c()), M, _dev(hist, torch.int32), _dev(base_slot_expert, torch.int32),
        _dev(slot_expert_mb, torch.int32), _dev(dev_status, torch.int32), _stream()))


def source_ids(shape: Shape, M: int, ids, tok_src, ids_v, dev_status=None) -> None:
    """(f.1) ids_v[L,T,K] = ids * M + tok_src[t] // (P // M): commodity (expert, source machine) ids."""
    _check("foremoe_source_ids", lib().foremoe_source_ids(
        C.byref(shape.c()), M, _dev(ids, torch.int32), _dev(tok_src, torch.int32),
        _dev(ids_v, torch.int32), _dev(dev_status, torch.int32), _stream()))


def local_placement(shape: Shape, M: int, slot_expert, slot_expert_v, dev_status=None) -> None:
    """(f.1) slot_expert [.,S] -> slot_expert_v [.,S*M]: allowed hosts of every commodity."""
    _check("foremoe_local_placement", lib().foremoe_local_placement(
        C.byref(shape.c()), M, _dev(slot_expert, torch.int32), _dev(slot_expert_v, torch.int32),
        _dev(dev_status, torch.int32), _stream()))


def traffic(shape: Shape, M: int, quota_v, traffic_out) -> None:
    """(f.1) quota_v [n_mb,L,S*M] -> traffic [n_mb,L,M,M] (Eq.(5) off the diagonal)."""
    _check("foremoe_traffic", lib().foremoe_traffic(
        C.byref(shape.c()), M, _dev(quota_v, torch.int32), _dev(traffic_out, torch.int32), _stream()))


def local_placement_theta(shape: Shape, M: int, num: int, den: int, hist_v, slot_expert, slot_expert_v_mb,
                          dev_status=None) -> None:
    """(f.1, C* term) one ladder member: hist_v [n_mb,L,E*M] + slot_expert -> slot_expert_v_mb [n_mb,L,S*M]."""
    _check("foremoe_local_placement_theta", lib().foremoe_local_placement_theta(
        C.byref(shape.c()), M, num, den, _dev(hist_v, torch.int32), _dev(slot_expert, torch.int32),
        _dev(slot_expert_v_mb, torch.int32), _dev(dev_status, torch.int32), _stream()))


def tradeoff_select(shape: Shape, M: int, a: int, b: int, rank_load_k, traffic_k, quota_k, slot_expert_v_k,
                    member, F, quota_sel, slot_expert_v_sel) -> None:
    """(f.1, C* term) per instance the member with the smallest a*L_max + b*C_max; [n_members, ...] inputs."""
    _check("foremoe_tradeoff_select", lib().foremoe_tradeoff_select(
        C.byref(shape.c()), M, int(rank_load_k.shape[0]), a, b, _dev(rank_load_k, torch.int32),
        _dev(traffic_k, torch.int32), _dev(quota_k, torch.int32), _dev(slot_expert_v_k, torch.int32),
        _dev(member, torch.int32), _dev(F, torch.int64), _dev(quota_sel, torch.int32),
        _dev(slot_expert_v_sel, torch.int32), _stream()))


def swap_relocation(shape: Shape, M: int, win: int, max_rounds: int, a: int, b: int, hist_v,
                    base_slot_expert, slot_expert_mb, rounds=None, dev_status=None) -> None:
    """(f.2) Alg. 2 Stage 2: hist_v [n_mb,L,E*M] + base [L,S] -> slot_expert_mb [n_mb,L,S]."""
    _check("foremoe_swap_relocation", lib().foremoe_swap_relocation(
        C.byref(shape.c()), M, win, max_rounds, a, b, _dev(hist_v, torch.int32),
        _dev(base_slot_expert, torch.int32), _dev(slot_expert_mb, torch.int32),
        _dev(rounds, torch.int32), _dev(dev_status, torch.int32), _stream()))


def replication(shape: Shape, M: int, hist, placed_slot_expert_mb, slot_expert_mb, dev_status=None) -> None:
    """(f.2) Stage 3 alone on per-micro-step placements with final base slots (may run in place)."""
    _check("foremoe_replication", lib().foremoe_replication(
        C.byref(shape.c()), M, _dev(hist, torch.int32), _dev(placed_slot_expert_mb, torch.int32),
        _dev(slot_expert_mb, torch.int32), _dev(dev_status, torch.int32), _stream()))


def replica_search(shape: Shape, M: int, max_copies: int, a: int, b: int, hist_v, placed_slot_expert_mb,
                   slot_expert_mb, replicas=None, F=None, dev_status=None) -> None:
    """(NEXT) Alg. 2 Stage 3: hist_v [n_mb,L,E*M] + placements with final base slots -> slot_expert_mb."""
    _check("foremoe_replica_search", lib().foremoe_replica_search(
        C.byref(shape.c()), M, max_copies, a, b, _dev(hist_v, torch.int32),
        _dev(placed_slot_expert_mb, torch.int32), _dev(slot_expert_mb, torch.int32),
        _dev(replicas, torch.int32), _dev(F, torch.int64), _dev(dev_status, torch.int32), _stream()))


def virtual_shape(shape: Shape, M: int) -> Shape:
    """Shape of the commodity instance: E, Nb, Nr (and the placement stride) multiplied by M."""
    return dataclasses.replace(shape, E=shape.E * M, Nb=shape.Nb * M, Nr=shape.Nr * M,
                               placement_mb_stride=shape.placement_mb_stride * M)


def step_host_arena_bytes(shape: Shape, mb_off_h) -> int:
    out = C.c_size_t(0)
    _check("foremoe_step_host_arena_bytes", lib().foremoe_step_host_arena_bytes(
        C.byref(shape.c()), _host(mb_off_h, torch.int32), C.byref(out)))
    return out.value


def step_host(shape: Shape, ids_h, w_h, mb_off_h, slot_expert_h, x_h, quota_h, rank_load_h,
              slot_off_h, y_h, arena, status_h) -> None:
    """The whole path from HOST tensors (pinned for speed); synchronises before returning."""
    _check("foremoe_step_host", lib().foremoe_step_host(
        C.byref(shape.c()), _host(ids_h, torch.int32), _host(w_h, torch.float32),
        _host(mb_off_h, torch.int32), _host(slot_expert_h, torch.int32),
        _host(x_h, shape.act_torch_dtype), _host(quota_h, torch.int32),
        _host(rank_load_h, torch.int32), _host(slot_off_h, torch.int32),
        _host(y_h, torch.float32), _dev(arena), arena.numel() * arena.element_size(),
        _host(status_h, torch.int32), _stream()))


def shape_of(cfg, T: Optional[int] = None, n_mb: Optional[int] = None, flags: int = 0) -> Shape:
    """Shape of a synth.TraceConfig."""
    return Shape(L=cfg.L, E=cfg.E, K=cfg.K, P=cfg.P, Nb=cfg.Nb, Nr=cfg.Nr,
                 T=cfg.T if T is None else T, n_mb=cfg.n_mb if n_mb is None else n_mb, H=cfg.H,
                 act_dtype=cfg.act_dtype, flags=flags)
