"""Thin ctypes binding of libppl (include/ppl.h): argument marshalling only.

Every step of the path (W-tile generation, (c,d) contraction, reduction/mirror) runs in the CUDA
kernels behind the C ABI.  PyTorch is used for FP64 device buffers and streams, nothing else.
There is no CPU fallback: if the library is missing or the device is not a B200-class GPU the
calls raise.  Function names mirror the C ABI (ppl_plan, ppl_apply, ppl_destroy, ...).
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, c_char_p, c_double, c_float, c_int, c_int32, c_size_t, c_uint64, c_void_p

from . import _build

PPL_OK = 0
PPL_ERR_INVALID_ARG = 1
PPL_ERR_WORKSPACE_TOO_SMALL = 2
PPL_ERR_ALLOC = 3
PPL_ERR_CUDA = 4
PPL_ERR_UNSUPPORTED_DEVICE = 5
PPL_ERR_PRECONDITION = 6
PPL_ERR_SCRATCH_LIMIT = 7
PPL_NOALLOC_SCRATCH_BYTES = 32 << 20  # include/ppl.h
PPL_SYM_NONE = 0
PPL_SYM_PAIR = 1
PPL_SYM_PAIR_SA = 2
PPL_SYM_FULL = 3
PPL_OPT_VERIFY_INPUTS = 1
PPL_LAYOUT_IJAB = 0
PPL_LAYOUT_IAJB = 1
LAYOUTS = {"ijab": PPL_LAYOUT_IJAB, "iajb": PPL_LAYOUT_IAJB}


class ppl_info_t(ctypes.Structure):
    _fields_ = [
        ("nocc", c_int32), ("nvirt", c_int32), ("nchol", c_int32), ("symmetry", c_int32),
        ("ta", c_int32), ("tb", c_int32), ("n_ablocks", c_int32), ("n_bblocks", c_int32),
        ("n_tiles", c_int32), ("ring", c_int32), ("splitk", c_int32), ("vec16", c_int32),
        ("launches_per_apply", c_int32), ("step1_tile_m", c_int32),
        ("workspace_bytes", c_uint64),
        ("flops_nominal", c_double), ("flops_executed", c_double),
        ("flops_step0", c_double), ("flops_step1", c_double),
        ("sa_splitk_plus", c_int32), ("sa_splitk_minus", c_int32),
        ("sa_tile_m_plus", c_int32), ("sa_tile_m_minus", c_int32),
        ("sa_rows_plus", c_int32), ("sa_rows_minus", c_int32),
        ("sa_k_plus", c_int32), ("sa_k_minus", c_int32),
        ("full_available", c_int32), ("full_tbg", c_int32), ("full_slabs", c_int32), ("full_tight", c_int32),
        ("full_workspace_bytes", c_uint64),
        ("flops_useful", c_double), ("flops_useful_step0", c_double), ("flops_useful_step1", c_double),
        ("small_fused", c_int32), ("reserved_", c_int32),
    ]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class ppl_times_t(ctypes.Structure):
    _fields_ = [
        ("total_ms", c_float), ("step0_ms", c_float), ("step1_ms", c_float), ("reduce_ms", c_float),
        ("n_step0", c_int32), ("n_step1", c_int32), ("n_reduce", c_int32),
        ("fold_ms", c_float), ("pack_ms", c_float), ("n_fold", c_int32), ("n_pack", c_int32),
    ]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class ppl_opts_t(ctypes.Structure):
    _fields_ = [("t2_layout", c_int32), ("r_layout", c_int32), ("alpha", c_double), ("beta", c_double)]


class ppl_debug_opts_t(ctypes.Structure):
    """include/ppl.h ppl_debug_opts_t: planner / orchestration knobs for tests and A/B runs; all zero = the defaults."""
    _fields_ = [(k, c_int32) for k in (
        "tile_edge", "ni_max", "cpasync_kernels", "full_min_v", "full_tbg", "full_slots", "full_strips", "full_tight",
        "full_rect_tiles", "full_no_diag_pack", "full_serial", "debug_sync", "trace", "host_chunk_mb", "no_small_fused", "host_panels", "full_group_m", "full_hints")] + [("reserved", c_int32 * 14)]


# Options merged under every Plan(...) / ppl_plan_dry(...) of this process.  Empty in the product; tests/conftest.py sets it so
# that the -m gpu tests of the TILED kernels keep running them at small shapes (the fused one-kernel path has its own tests).
DEFAULT_DEBUG: dict = {}


def _debug_opts(debug):
    debug = {**DEFAULT_DEBUG, **(debug or {})}
    if not debug:
        return None
    d = ppl_debug_opts_t()
    names = {k for k, _ in ppl_debug_opts_t._fields_} - {"reserved"}
    for k, val in debug.items():
        if k not in names:
            raise KeyError(f"unknown debug option {k!r}; known: {sorted(names)}")
        setattr(d, k, int(val))
    return ctypes.byref(d)


class PplError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {error_string(code)} (PPL error {code})")


# Every symbol include/ppl.h declares: (restype, argtypes)
SYMBOLS = {
    "ppl_plan": (c_void_p, [c_int, c_int, c_int, c_size_t]),
    "ppl_plan_ex": (c_void_p, [c_int, c_int, c_int, c_size_t, POINTER(ppl_debug_opts_t)]),
    "ppl_apply": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "ppl_apply_ex": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, POINTER(ppl_opts_t), c_void_p]),
    "ppl_apply_dense": (c_int, [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, POINTER(ppl_opts_t), c_void_p]),
    "ppl_generate_eri": (c_int, [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p]),
    "ppl_contract_pair_workspace": (c_int, [c_char_p, POINTER(ctypes.c_int64), POINTER(ctypes.c_int64), POINTER(c_size_t)]),
    "ppl_contract_pair": (c_int, [c_char_p, POINTER(ctypes.c_int64), POINTER(ctypes.c_int64), c_void_p, c_void_p, c_void_p,
                                  c_double, c_double, c_void_p, c_size_t, c_void_p]),
    "ppl_contract_pair_noalloc": (c_int, [c_char_p, POINTER(ctypes.c_int64), POINTER(ctypes.c_int64), c_void_p, c_void_p, c_void_p,
                                          c_double, c_double, c_void_p]),
    "ppl_apply_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, POINTER(c_uint64), POINTER(c_uint64)]),
    "ppl_apply_profiled": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, POINTER(ppl_times_t)]),
    "ppl_destroy": (c_int, [c_void_p]),
    "ppl_last_error": (c_int, []),
    "ppl_error_string": (c_char_p, [c_int]),
    "ppl_plan_set_symmetry": (c_int, [c_void_p, c_int]),
    "ppl_plan_set_graph": (c_int, [c_void_p, c_int]),
    "ppl_plan_set_option": (c_int, [c_void_p, c_int, c_int]),
    "ppl_plan_verify_status": (c_int, [c_void_p, POINTER(c_int)]),
    "ppl_plan_info": (c_int, [c_void_p, POINTER(ppl_info_t)]),
    "ppl_plan_dry": (c_int, [c_int, c_int, c_int, c_size_t, c_size_t, c_int, c_int, POINTER(ppl_info_t)]),
    "ppl_plan_dry_ex": (c_int, [c_int, c_int, c_int, c_size_t, c_size_t, c_int, c_int, POINTER(ppl_debug_opts_t), POINTER(ppl_info_t)]),
    "ppl_check_inputs": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, POINTER(c_int)]),
    "ppl_probe_fp64_peak": (c_int, [POINTER(c_double), c_int, c_double]),
    "ppl_probe_fp64_pipe": (c_int, [c_int, POINTER(c_double), c_int, c_double]),
    "ppl_debug_dmma_layout": (c_int, [c_void_p, c_void_p, c_void_p]),
}

_lib = None


def lib() -> ctypes.CDLL:
    """Load libppl.so (building it in-tree with nvcc if stale).  Raises if that is impossible."""
    global _lib
    if _lib is None:
        so = _build.build()
        L = ctypes.CDLL(so)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)  # AttributeError if the ABI is incomplete
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def library_path() -> str:
    return _build.SO


def error_string(code: int) -> str:
    return lib().ppl_error_string(code).decode()


def ppl_last_error() -> int:
    return int(lib().ppl_last_error())


def _check(rc: int, where: str):
    if rc != PPL_OK:
        raise PplError(rc, where)


def _dev_ptr(t, name: str, shape=None):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: need a contiguous CUDA float64 tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return c_void_p(t.data_ptr())


def _stream_ptr(stream):
    import torch

    if stream is None:
        stream = torch.cuda.current_stream()
    return c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


class Plan:
    """Owner of an opaque ppl_plan_t* (workspace, internal stream, events)."""

    def __init__(self, nocc: int, nvirt: int, nchol: int, workspace_bytes: int = 0, debug: dict | None = None):
        """debug: ppl_debug_opts_t fields by name (tests / A-B runs only); None = ppl_plan."""
        if debug or DEFAULT_DEBUG:
            h = lib().ppl_plan_ex(int(nocc), int(nvirt), int(nchol), int(workspace_bytes), _debug_opts(debug))
        else:
            h = lib().ppl_plan(int(nocc), int(nvirt), int(nchol), int(workspace_bytes))
        if not h:
            raise PplError(ppl_last_error(), "ppl_plan")
        self._h = c_void_p(h)
        self.nocc, self.nvirt, self.nchol = int(nocc), int(nvirt), int(nchol)

    # -- C ABI mirrors -------------------------------------------------------------------------
    def apply(self, L, t2, R, stream=None):
        """R += ladder(L, t2), asynchronously on `stream` (default: torch's current stream)."""
        o, v, x = self.nocc, self.nvirt, self.nchol
        _check(lib().ppl_apply(self._h, _dev_ptr(L, "L", (x, v, v)), _dev_ptr(t2, "t2", (o, o, v, v)),
                               _dev_ptr(R, "R", (o, o, v, v)), _stream_ptr(stream)), "ppl_apply")
        return R

    def _shape4(self, layout: str):
        o, v = self.nocc, self.nvirt
        return (o, o, v, v) if layout == "ijab" else (o, v, o, v)

    def apply_ex(self, L, t2, R, t2_layout="ijab", r_layout="ijab", alpha=1.0, beta=1.0, stream=None):
        """R = beta*R + alpha*ladder(L, t2); t2 / R stored 'ijab' ([i,j,c,d]) or 'iajb' ([i,c,j,d])."""
        v, x = self.nvirt, self.nchol
        opts = ppl_opts_t(LAYOUTS[t2_layout], LAYOUTS[r_layout], float(alpha), float(beta))
        _check(lib().ppl_apply_ex(self._h, _dev_ptr(L, "L", (x, v, v)), _dev_ptr(t2, "t2", self._shape4(t2_layout)),
                                  _dev_ptr(R, "R", self._shape4(r_layout)), ctypes.byref(opts), _stream_ptr(stream)),
               "ppl_apply_ex")
        return R

    def apply_dense(self, eri, a0, t2, R, t2_layout="ijab", r_layout="ijab", alpha=1.0, beta=1.0, stream=None):
        """Step 1 alone on a dense slab eri[na][v][v][v] of <ab|cd>, a0 <= a < a0+na (the paper's 'abcd,ecfd->efab')."""
        v = self.nvirt
        na = int(eri.shape[0])
        opts = ppl_opts_t(LAYOUTS[t2_layout], LAYOUTS[r_layout], float(alpha), float(beta))
        _check(lib().ppl_apply_dense(self._h, _dev_ptr(eri, "eri", (na, v, v, v)), int(a0), na,
                                     _dev_ptr(t2, "t2", self._shape4(t2_layout)), _dev_ptr(R, "R", self._shape4(r_layout)),
                                     ctypes.byref(opts), _stream_ptr(stream)), "ppl_apply_dense")
        return R

    def generate_eri(self, L, a0, na, eri, stream=None):
        """Step 0 alone: eri[na][v][v][v] = <ab|cd> for a0 <= a < a0+na (the paper's 'xac,xbd->acbd' in 'abcd' order)."""
        v, x = self.nvirt, self.nchol
        _check(lib().ppl_generate_eri(self._h, _dev_ptr(L, "L", (x, v, v)), int(a0), int(na),
                                      _dev_ptr(eri, "eri", (int(na), v, v, v)), _stream_ptr(stream)), "ppl_generate_eri")
        return eri

    def apply_profiled(self, L, t2, R, stream=None) -> dict:
        o, v, x = self.nocc, self.nvirt, self.nchol
        t = ppl_times_t()
        _check(lib().ppl_apply_profiled(self._h, _dev_ptr(L, "L", (x, v, v)), _dev_ptr(t2, "t2", (o, o, v, v)),
                                        _dev_ptr(R, "R", (o, o, v, v)), _stream_ptr(stream), ctypes.byref(t)),
               "ppl_apply_profiled")
        return t.asdict()

    def apply_host(self, L, t2, R):
        """Host (numpy float64 / CPU torch) buffers; copies are part of the call. Returns (h2d, d2h) bytes."""
        o, v, x = self.nocc, self.nvirt, self.nchol

        def hp(a, name, shape):
            import numpy as np

            if hasattr(a, "data_ptr"):  # CPU torch tensor (e.g. pinned)
                import torch

                if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or tuple(a.shape) != shape:
                    raise TypeError(f"{name}: need a contiguous CPU float64 tensor of shape {shape}")
                return c_void_p(a.data_ptr())
            if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous or a.shape != shape:
                raise TypeError(f"{name}: need a C-contiguous float64 array of shape {shape}")
            return c_void_p(a.ctypes.data)

        h2d, d2h = c_uint64(0), c_uint64(0)
        _check(lib().ppl_apply_host(self._h, hp(L, "L", (x, v, v)), hp(t2, "t2", (o, o, v, v)),
                                    hp(R, "R", (o, o, v, v)), ctypes.byref(h2d), ctypes.byref(d2h)), "ppl_apply_host")
        return int(h2d.value), int(d2h.value)

    def set_symmetry(self, mode: int):
        _check(lib().ppl_plan_set_symmetry(self._h, int(mode)), "ppl_plan_set_symmetry")

    def set_graph(self, mode: int):
        """-1 auto (default), 0 plain launches, 1 replay one CUDA graph per (L, t2, R, opts) key."""
        _check(lib().ppl_plan_set_graph(self._h, int(mode)), "ppl_plan_set_graph")

    def set_verify(self, mode: int):
        """PPL_OPT_VERIFY_INPUTS: 1 (default) check at the head of every apply, reported by the next call; 2 synchronous; 0 off."""
        _check(lib().ppl_plan_set_option(self._h, PPL_OPT_VERIFY_INPUTS, int(mode)), "ppl_plan_set_option")

    def verify_status(self) -> int:
        """Waits for the pending check of the last apply; returns its flags, raises PplError(PPL_ERR_PRECONDITION) on a violation."""
        flags = c_int(0)
        rc = lib().ppl_plan_verify_status(self._h, ctypes.byref(flags))
        if rc != PPL_OK:
            raise PplError(rc, "ppl_plan_verify_status")
        return int(flags.value)

    def info(self) -> dict:
        out = ppl_info_t()
        _check(lib().ppl_plan_info(self._h, ctypes.byref(out)), "ppl_plan_info")
        return out.asdict()

    def check_inputs(self, L, t2, stream=None) -> int:
        """Returns flags (bit 0: L not symmetric, bit 1: t2 not pair-symmetric); raises on a violated precondition."""
        flags = c_int(0)
        rc = lib().ppl_check_inputs(self._h, _dev_ptr(L, "L"), _dev_ptr(t2, "t2"), _stream_ptr(stream), ctypes.byref(flags))
        if rc not in (PPL_OK, PPL_ERR_PRECONDITION):
            raise PplError(rc, "ppl_check_inputs")
        if rc == PPL_ERR_PRECONDITION:
            raise PplError(rc, "ppl_check_inputs")
        return int(flags.value)

    def destroy(self):
        if self._h:
            rc = lib().ppl_destroy(self._h)
            self._h = c_void_p(None)
            _check(rc, "ppl_destroy")

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        if exc[0] is None:
            self.destroy()
            return
        try:  # an exception is already on its way out of the with-block: a late PPL_ERR_PRECONDITION must not mask it
            self.destroy()
        except PplError:
            pass

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# function-style mirrors of the three north_star entry points
def ppl_plan(nocc: int, nvirt: int, nchol: int, workspace_bytes: int = 0) -> Plan:
    return Plan(nocc, nvirt, nchol, workspace_bytes)


def ppl_plan_dry(nocc: int, nvirt: int, nchol: int, workspace_bytes: int = 0, device_free_bytes: int = 170 << 30,
                 num_sms: int = 148, mode: int = -1, debug: dict | None = None) -> dict:
    """The planner alone, for a stated device: no GPU needed.  Returns what Plan.info() would."""
    out = ppl_info_t()
    _check(lib().ppl_plan_dry_ex(int(nocc), int(nvirt), int(nchol), int(workspace_bytes), int(device_free_bytes), int(num_sms),
                                 int(mode), _debug_opts(debug), ctypes.byref(out)), "ppl_plan_dry")
    return out.asdict()


def ppl_apply(plan: Plan, L, t2, R, stream=None):
    return plan.apply(L, t2, R, stream)


def ppl_destroy(plan: Plan):
    plan.destroy()


def ppl_probe_fp64_peak(reps: int = 3, ms_target: float = 20.0) -> float:
    out = c_double(0.0)
    _check(lib().ppl_probe_fp64_peak(ctypes.byref(out), int(reps), float(ms_target)), "ppl_probe_fp64_peak")
    return float(out.value)


def ppl_contract_pair(subscripts: str, A, B, C=None, alpha: float = 1.0, beta: float = 0.0, stream=None, workspace=None):
    """C = beta*C + alpha*einsum(subscripts, A, B) for a two-operand contraction of tensordot type (include/ppl.h).
    A, B, C: contiguous CUDA float64 tensors; C=None allocates the output (beta is then 0).  The workspace (a torch
    uint8 CUDA tensor) is allocated per call unless one is passed in; it must outlive the queued work."""
    import torch

    ins, out = subscripts.replace(" ", "").split("->")
    s0, s1 = ins.split(",")
    d0 = (ctypes.c_int64 * max(A.dim(), 1))(*A.shape)
    d1 = (ctypes.c_int64 * max(B.dim(), 1))(*B.shape)
    ext = dict(zip(s0, A.shape))
    ext.update(zip(s1, B.shape))
    shape = tuple(ext[c] for c in out)
    if C is None:
        C, beta = torch.empty(shape, dtype=torch.float64, device=A.device), 0.0
    need = c_size_t(0)
    _check(lib().ppl_contract_pair_workspace(subscripts.encode(), d0, d1, ctypes.byref(need)), "ppl_contract_pair_workspace")
    if workspace is None:
        workspace = torch.empty(int(need.value) + 256, dtype=torch.uint8, device=A.device)
    base = workspace.data_ptr()
    aligned = (base + 255) // 256 * 256
    _check(lib().ppl_contract_pair(subscripts.encode(), d0, d1, _dev_ptr(A, "A"), _dev_ptr(B, "B"), _dev_ptr(C, "C", shape),
                                   float(alpha), float(beta), c_void_p(aligned), workspace.numel() - (aligned - base),
                                   _stream_ptr(stream)), "ppl_contract_pair")
    if hasattr(workspace, "record_stream"):
        workspace.record_stream(stream if stream is not None else torch.cuda.current_stream())
    return C


def ppl_contract_pair_noalloc(subscripts: str, A, B, C, alpha: float = 1.0, beta: float = 0.0, stream=None):
    """C = beta*C + alpha*einsum(subscripts, A, B) through the entry point that allocates nothing (include/ppl.h).

    For callers that cannot get device memory of their own -- the GPU already belongs to someone's pool, or the call sits
    where cudaMalloc's device-wide synchronisation is not acceptable.  Accordingly this wrapper allocates nothing either: the
    caller passes the output C (a contiguous CUDA float64 tensor of the shape `out` spells), and there is no workspace
    argument -- the library's fixed 32 MiB array (PPL_NOALLOC_SCRATCH_BYTES, one per GPU, shared by all calls) is the scratch.
    Raises PplError(PPL_ERR_SCRATCH_LIMIT) when the request's offset tables do not fit into it.  Calls that may overlap on
    the GPU (different streams, no ordering) race on that array; keep them on one stream."""
    ins, out = subscripts.replace(" ", "").split("->")
    s0, s1 = ins.split(",")
    d0 = (ctypes.c_int64 * max(A.dim(), 1))(*A.shape)
    d1 = (ctypes.c_int64 * max(B.dim(), 1))(*B.shape)
    ext = dict(zip(s0, A.shape))
    ext.update(zip(s1, B.shape))
    shape = tuple(ext[c] for c in out)
    _check(lib().ppl_contract_pair_noalloc(subscripts.encode(), d0, d1, _dev_ptr(A, "A"), _dev_ptr(B, "B"), _dev_ptr(C, "C", shape),
                                           float(alpha), float(beta), _stream_ptr(stream)), "ppl_contract_pair_noalloc")
    return C


PROBE_KINDS = {"dmma8": 0, "dmma16": 1, "dfma16": 2, "mix8": 3}


def ppl_probe_fp64_pipe(kind: str, reps: int = 3, ms_target: float = 20.0) -> float:
    """TFLOP/s of a register-only instruction stream: 'dmma8' (the peak probe), 'dmma16', 'dfma16', 'mix8'."""
    out = c_double(0.0)
    _check(lib().ppl_probe_fp64_pipe(PROBE_KINDS[kind], ctypes.byref(out), int(reps), float(ms_target)), "ppl_probe_fp64_pipe")
    return float(out.value)


def ppl_debug_dmma_layout(A, B, C):
    _check(lib().ppl_debug_dmma_layout(_dev_ptr(A, "A", (8, 4)), _dev_ptr(B, "B", (4, 8)), _dev_ptr(C, "C", (8, 8))),
           "ppl_debug_dmma_layout")
    return C
