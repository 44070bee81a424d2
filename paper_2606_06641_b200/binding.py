"""Thin ctypes binding over the C ABI of include/afsat.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libafsat_b200.so; PyTorch is used for
device memory and streams.  There is NO CPU fallback: if the shared library is missing or no
CUDA device is usable, the calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libafsat_b200.so"
_lib = None

FLAG_DEFAULT = 0
FLAG_ROBUST = 1
FLAG_PAPER = 2
MAX_LEN = 64
STEP_AUTO, STEP_LAUNCHES, STEP_PERSISTENT, STEP_GRAPH = range(4)

Q_KERNEL_LAUNCHES, Q_NUM_SIGNATURES, Q_NUM_BUCKETS, Q_NNZ, Q_WORKSPACE_BYTES, Q_SM_COUNT, \
    Q_FP_INSTR_PER_CANDIDATE, Q_PROFILED_EVAL_NS, Q_PROFILED_EVAL_LAUNCHES, Q_FLOP_PER_CANDIDATE, Q_NUM_GROUPS, \
    Q_STEP_PATH, Q_TILE_W, Q_LIVE_CONSTRAINTS, Q_LIVE_NNZ, Q_DECIDED_SATISFIED, Q_L2_BYTES, Q_PROFILED_UPDATE_NS, \
    Q_PROFILED_CHECK_NS = range(19)

ERROR_NAMES = {0: "AFSAT_OK", -1: "AFSAT_E_INVALID", -2: "AFSAT_E_LENGTH", -3: "AFSAT_E_VARIABLE",
               -4: "AFSAT_E_SIGN", -5: "AFSAT_E_DUPLICATE", -6: "AFSAT_E_PARAM",
               -7: "AFSAT_E_NOMEM", -8: "AFSAT_E_CUDA", -9: "AFSAT_E_UNSAT"}

STATIC_SCRATCH_BYTES = 8 << 20      # AFSAT_STATIC_SCRATCH_BYTES of include/afsat.h

EXPORTS = ["afsat_static_setup", "afsat_check_static", "afsat_create", "afsat_create_ex", "afsat_probe_peak", "afsat_host_restrict", "afsat_host_tables_mask", "afsat_destroy", "afsat_last_error", "afsat_eval_grad", "afsat_check",
           "afsat_step", "afsat_step_host", "afsat_host_tables", "afsat_query", "afsat_version",
           "afsat_set_profiling", "afsat_step_ls", "afsat_parse", "afsat_parse_file", "afsat_parse_error",
           "afsat_problem_sizes", "afsat_problem_fill", "afsat_problem_free", "afsat_restart", "afsat_solve"]


class Options(C.Structure):
    """struct afsat_options of include/afsat.h."""
    _fields_ = [("struct_size", C.c_uint32), ("flags", C.c_uint32), ("n_groups", C.c_int32), ("step_path", C.c_int32),
                ("tile_w", C.c_int64), ("l2_budget_bytes", C.c_int64)]


class AfsatError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {message}")
        self.code = code


def load_library():
    """dlopen the in-tree CUDA library; raises (loudly) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise ImportError(f"{LIB_PATH} is missing: build it with "
                          f"`python -m paper_2606_06641_b200.build` (no CPU fallback exists)")
    L = C.CDLL(str(LIB_PATH))
    vp, i32, i64, u32, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_double
    L.afsat_create.restype = C.c_int
    L.afsat_create.argtypes = [C.POINTER(vp), i32, i32, vp, vp, vp, vp, vp, vp, i32, i64, i32, i32, u32]
    L.afsat_create_ex.restype = C.c_int
    L.afsat_create_ex.argtypes = [C.POINTER(vp), i32, i32, vp, vp, vp, vp, vp, vp, i32, i64, i32, i32, C.POINTER(Options)]
    L.afsat_probe_peak.restype = C.c_int
    L.afsat_probe_peak.argtypes = [i32, i32, C.POINTER(dbl)]
    L.afsat_destroy.restype = None
    L.afsat_destroy.argtypes = [vp]
    L.afsat_last_error.restype = C.c_char_p
    L.afsat_last_error.argtypes = [vp]
    L.afsat_eval_grad.restype = C.c_int
    L.afsat_eval_grad.argtypes = [vp, vp, vp, vp, vp]
    L.afsat_check.restype = C.c_int
    L.afsat_check.argtypes = [vp, vp, vp, vp, vp]
    L.afsat_static_setup.restype = C.c_int
    L.afsat_static_setup.argtypes = [i32]
    L.afsat_check_static.restype = C.c_int
    L.afsat_check_static.argtypes = [vp, vp, vp, vp, vp]
    L.afsat_step.restype = C.c_int
    L.afsat_step.argtypes = [vp, vp, dbl, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    L.afsat_step_ls.restype = C.c_int
    L.afsat_step_ls.argtypes = [vp, vp, dbl, dbl, dbl, dbl, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
    L.afsat_restart.restype = C.c_int
    L.afsat_restart.argtypes = [vp, vp, vp, C.c_uint64, u32, vp]
    L.afsat_solve.restype = C.c_int
    L.afsat_solve.argtypes = [vp, vp, dbl, i32, i32, C.c_uint64, i32, vp, vp, vp, vp, vp, vp]
    L.afsat_step_host.restype = C.c_int
    L.afsat_step_host.argtypes = [vp, vp, dbl, i32, vp, vp, vp, vp, vp]
    L.afsat_host_tables.restype = C.c_int
    L.afsat_host_tables.argtypes = [i32, i32, i32, u32, vp, vp]
    L.afsat_host_restrict.restype = C.c_int
    L.afsat_host_restrict.argtypes = [i32, i32, i32, i32, i32, vp, vp]
    L.afsat_host_tables_mask.restype = C.c_int
    L.afsat_host_tables_mask.argtypes = [i32, C.c_uint64, C.c_uint64, u32, vp, vp]
    L.afsat_query.restype = i64
    L.afsat_query.argtypes = [vp, i32]
    L.afsat_set_profiling.restype = C.c_int
    L.afsat_set_profiling.argtypes = [vp, i32]
    L.afsat_parse.restype = C.c_int
    L.afsat_parse.argtypes = [C.c_char_p, i64, C.POINTER(vp)]
    L.afsat_parse_file.restype = C.c_int
    L.afsat_parse_file.argtypes = [C.c_char_p, C.POINTER(vp)]
    L.afsat_parse_error.restype = C.c_char_p
    L.afsat_parse_error.argtypes = []
    L.afsat_problem_sizes.restype = C.c_int
    L.afsat_problem_sizes.argtypes = [vp, vp, vp, vp, vp]
    L.afsat_problem_fill.restype = C.c_int
    L.afsat_problem_fill.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.afsat_problem_free.restype = None
    L.afsat_problem_free.argtypes = [vp]
    L.afsat_version.restype = C.c_char_p
    L.afsat_version.argtypes = []
    _lib = L
    return L


def version() -> str:
    return load_library().afsat_version().decode()


def probe_peak(kind: int, device: int = 0) -> float:
    """afsat_probe_peak: measured TFLOP/s of independent FMA chains; kind 0 = FFMA, 1 = FFMA2, 2 = DFMA."""
    L = load_library()
    out = C.c_double(0.0)
    rc = L.afsat_probe_peak(int(device), int(kind), C.byref(out))
    if rc != 0:
        raise AfsatError(rc, L.afsat_last_error(None).decode())
    return float(out.value)


def static_setup(device: int = 0) -> None:
    """afsat_static_setup: resolve the device address of the library's static scratch array on `device` (once per
    device, at set-up; before any graph capture)."""
    L = load_library()
    rc = L.afsat_static_setup(int(device))
    if rc != 0:
        raise AfsatError(rc, L.afsat_last_error(None).decode())


def host_tables(ctype: int, k: int, param: int, flags: int = 0):
    """(rows [P,8] float64, n_real) -- see afsat_host_tables in include/afsat.h.  Host only."""
    L = load_library()
    tab = np.zeros((MAX_LEN // 2 + 1, 8), dtype=np.float64)
    n_real = C.c_int32(0)
    rc = L.afsat_host_tables(ctype, k, param, flags, tab.ctypes.data, C.addressof(n_real))
    if rc < 0:
        raise AfsatError(rc, "afsat_host_tables")
    return tab[:rc].copy(), int(n_real.value)


def host_restrict(ctype: int, k: int, param: int, f_true: int, f_false: int):
    """afsat_host_restrict: (status, k_free, mask) of a constraint under a partial assignment; status 0 = still depends on
    its free literals, 1 = satisfied, 2 = violated; mask = Python int with bit tau' set iff tau' free true literals satisfy."""
    L = load_library()
    kf = C.c_int32(0)
    mk = (C.c_uint64 * 2)(0, 0)
    rc = L.afsat_host_restrict(ctype, k, param, f_true, f_false, C.addressof(kf), C.addressof(mk))
    if rc < 0:
        raise AfsatError(rc, "afsat_host_restrict")
    return rc, int(kf.value), int(mk[0]) | (int(mk[1]) << 64)


def host_tables_mask(k: int, mask: int, flags: int = 0):
    """(rows [P,8] float64, n_real) of the signature (k literals, satisfying counts = bits of mask).  Host only."""
    L = load_library()
    tab = np.zeros((MAX_LEN // 2 + 1, 8), dtype=np.float64)
    n_real = C.c_int32(0)
    rc = L.afsat_host_tables_mask(k, mask & 0xFFFFFFFFFFFFFFFF, mask >> 64, flags, tab.ctypes.data, C.addressof(n_real))
    if rc < 0:
        raise AfsatError(rc, "afsat_host_tables_mask")
    return tab[:rc].copy(), int(n_real.value)


class Problem:
    """What afsat_parse produced: the CSR constraint table and the partial-assignment mask (numpy)."""

    def __init__(self, n_vars, row_ptr, lit_var, lit_sign, ctype, param, fixed, stats):
        self.n_vars, self.row_ptr, self.lit_var, self.lit_sign = n_vars, row_ptr, lit_var, lit_sign
        self.ctype, self.param, self.fixed, self.stats = ctype, param, fixed, stats
        self.n_cons = int(row_ptr.shape[0] - 1)

    def context(self, *, batch, dtype=32, device=0, flags=0, ldb=None, **opts):
        return Context(self.n_vars, self.row_ptr, self.lit_var, self.lit_sign, self.ctype, self.param,
                       self.fixed, batch=batch, ldb=ldb, dtype=dtype, device=device, flags=flags, **opts)


def _take_problem(L, rc, h):
    if rc != 0:
        raise AfsatError(rc, L.afsat_parse_error().decode())
    try:
        n, m, nnz = C.c_int32(0), C.c_int32(0), C.c_int64(0)
        stats = np.zeros(5, dtype=np.int64)
        L.afsat_problem_sizes(h, C.addressof(n), C.addressof(m), C.addressof(nnz), stats.ctypes.data)
        row_ptr = np.zeros(m.value + 1, dtype=np.int64)
        lit_var = np.zeros(nnz.value, dtype=np.int32)
        lit_sign = np.zeros(nnz.value, dtype=np.int8)
        ctype = np.zeros(m.value, dtype=np.uint8)
        param = np.zeros(m.value, dtype=np.int32)
        fixed = np.zeros(n.value, dtype=np.int8)
        rc = L.afsat_problem_fill(h, row_ptr.ctypes.data, lit_var.ctypes.data if nnz.value else None,
                                  lit_sign.ctypes.data if nnz.value else None,
                                  ctype.ctypes.data if m.value else None, param.ctypes.data if m.value else None,
                                  fixed.ctypes.data)
        if rc != 0:
            raise AfsatError(rc, "afsat_problem_fill")
        names = ("constraints_read", "variables_assigned", "constraints_discarded", "declared_vars", "declared_constraints")
        return Problem(int(n.value), row_ptr, lit_var, lit_sign, ctype, param, fixed, dict(zip(names, stats.tolist())))
    finally:
        L.afsat_problem_free(h)


def parse(text) -> Problem:
    """afsat_parse: DIMACS CNF / hybrid PB text (str or bytes) -> Problem.  Host only."""
    L = load_library()
    data = text.encode() if isinstance(text, str) else bytes(text)
    h = C.c_void_p(None)
    rc = L.afsat_parse(data, len(data), C.byref(h))
    return _take_problem(L, rc, h)


def parse_file(path) -> Problem:
    L = load_library()
    h = C.c_void_p(None)
    rc = L.afsat_parse_file(str(path).encode(), C.byref(h))
    return _take_problem(L, rc, h)


def _np_ptr(a):
    return None if a is None else a.ctypes.data


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


class Context:
    """An afsat_ctx for one instance.  Tensors are torch CUDA tensors, variable-major [n, ldb]."""

    def __init__(self, n_vars, row_ptr, lit_var, lit_sign, ctype, param, fixed=None, *, batch,
                 ldb=None, dtype=32, device=0, flags=0, tile_w=0, l2_budget_bytes=0, step_path=STEP_AUTO):
        """fixed: None, [n] (one partial assignment) or [n_groups, n] (several; afsat_create_ex)."""
        L = load_library()
        self._L = L
        self._h = C.c_void_p(None)
        row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
        lit_var = np.ascontiguousarray(lit_var, dtype=np.int32)
        lit_sign = np.ascontiguousarray(lit_sign, dtype=np.int8)
        ctype = np.ascontiguousarray(ctype, dtype=np.uint8)
        param = np.ascontiguousarray(param, dtype=np.int32)
        fixed = None if fixed is None else np.ascontiguousarray(fixed, dtype=np.int8)
        self.n_groups = 1 if fixed is None or fixed.ndim == 1 else int(fixed.shape[0])
        self.n = int(n_vars)
        self.m = int(row_ptr.shape[0] - 1)
        self.B = int(batch)
        self.ldb = int(ldb) if ldb is not None else (self.B + 31) // 32 * 32
        self.dtype = int(dtype)
        self.device = int(device)
        if self.n_groups == 1 and not tile_w and not l2_budget_bytes and step_path == STEP_AUTO:
            rc = L.afsat_create(C.byref(self._h), self.n, self.m, _np_ptr(row_ptr), _np_ptr(lit_var),
                                _np_ptr(lit_sign), _np_ptr(ctype), _np_ptr(param), _np_ptr(fixed),
                                self.B, self.ldb, self.dtype, self.device, int(flags))
        else:
            opt = Options(C.sizeof(Options), int(flags), self.n_groups, int(step_path), int(tile_w), int(l2_budget_bytes))
            rc = L.afsat_create_ex(C.byref(self._h), self.n, self.m, _np_ptr(row_ptr), _np_ptr(lit_var),
                                   _np_ptr(lit_sign), _np_ptr(ctype), _np_ptr(param), _np_ptr(fixed),
                                   self.B, self.ldb, self.dtype, self.device, C.byref(opt))
        if rc != 0:
            msg = L.afsat_last_error(None).decode()
            self._h = C.c_void_p(None)
            raise AfsatError(rc, msg)

    @classmethod
    def from_instance(cls, inst, *, batch=None, dtype=32, device=0, flags=0, ldb=None, fixed="instance", **opts):
        return cls(inst.n_vars, inst.row_ptr, inst.lit_var, inst.lit_sign, inst.ctype, inst.param,
                   inst.fixed if isinstance(fixed, str) else fixed,
                   batch=int(batch if batch is not None else inst.batch), ldb=ldb,
                   dtype=dtype, device=device, flags=flags, **opts)

    # ---- helpers -------------------------------------------------------------------------
    def _torch_dtype(self):
        import torch
        return torch.float32 if self.dtype == 32 else torch.float64

    def _check_x(self, x):
        import torch
        if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == self._torch_dtype()
                and x.is_contiguous() and tuple(x.shape) == (self.n, self.ldb)
                and x.device.index == self.device):
            raise ValueError(f"expected a contiguous CUDA tensor [{self.n},{self.ldb}] "
                             f"{self._torch_dtype()} on device {self.device}")

    def _raise(self, rc):
        if rc != 0:
            raise AfsatError(rc, self._L.afsat_last_error(self._h).decode())

    def new_tensor(self, fill=None):
        import torch
        return torch.zeros((self.n, self.ldb), dtype=self._torch_dtype(), device=f"cuda:{self.device}")

    # ---- entry points (same names as the C ABI) ---------------------------------------------
    def eval_grad(self, x, F=None, G=None, *, want_F=True, want_G=True, stream=None):
        import torch
        self._check_x(x)
        dev = x.device
        if want_F and F is None:
            F = torch.empty(self.B, dtype=x.dtype, device=dev)
        if want_G and G is None:
            G = torch.empty_like(x)
        if G is not None:
            self._check_x(G)
        rc = self._L.afsat_eval_grad(self._h, x.data_ptr(), F.data_ptr() if F is not None else None,
                                     G.data_ptr() if G is not None else None, _stream_ptr(stream))
        self._raise(rc)
        return F, G

    def check(self, x, sat_count=None, is_solution=None, *, stream=None):
        import torch
        self._check_x(x)
        if sat_count is None:
            sat_count = torch.empty(self.B, dtype=torch.int32, device=x.device)
        if is_solution is None:
            is_solution = torch.empty(self.B, dtype=torch.uint8, device=x.device)
        rc = self._L.afsat_check(self._h, x.data_ptr(), sat_count.data_ptr(), is_solution.data_ptr(),
                                 _stream_ptr(stream))
        self._raise(rc)
        return sat_count, is_solution

    def check_static(self, x, sat_count, is_solution, *, stream=None):
        """afsat_check_static: the check with its scratch in the library's static device array -- the call allocates
        nothing, so the caller passes the outputs too ([B] int32, [B] uint8 CUDA tensors).  All calls on a device share
        the array: order them on the GPU."""
        self._check_x(x)
        rc = self._L.afsat_check_static(self._h, x.data_ptr(), sat_count.data_ptr(), is_solution.data_ptr(),
                                        _stream_ptr(stream))
        self._raise(rc)
        return sat_count, is_solution

    def step(self, x, eta, n_steps, *, step_base=0, state=None, want_F=True, F=None, F_pre=None,
             h_any_solved=None, stream=None):
        """In-place n_steps of PGD on x.  Returns (F, sat_count, is_solution, first_step); F_pre (a [B] tensor, optional)
        receives F(X(n_steps - 1)), the by-product of the last fused gradient pass."""
        import torch
        self._check_x(x)
        dev = x.device
        if want_F and F is None:
            F = torch.empty(self.B, dtype=x.dtype, device=dev)
        sat = torch.empty(self.B, dtype=torch.int32, device=dev)
        if state is None:
            sol = torch.empty(self.B, dtype=torch.uint8, device=dev)
            first = torch.empty(self.B, dtype=torch.int32, device=dev)
            resume = 0
        else:
            sol, first = state
            resume = 1
        hp = None
        if h_any_solved is not None:
            assert h_any_solved.is_pinned() and h_any_solved.dtype == torch.int32 and h_any_solved.numel() >= 2
            hp = h_any_solved.data_ptr()
        rc = self._L.afsat_step(self._h, x.data_ptr(), float(eta), int(n_steps), int(step_base), resume,
                                F.data_ptr() if F is not None else None,
                                F_pre.data_ptr() if F_pre is not None else None, sat.data_ptr(), sol.data_ptr(),
                                first.data_ptr(), hp, _stream_ptr(stream))
        self._raise(rc)
        return F, sat, sol, first

    def step_ls(self, x, n_steps, *, s_max=1.0, beta=0.5, c1=1e-4, delta=1e-6, max_trials=8, step_base=0,
                state=None, want_F=True, h_any_solved=None, stream=None):
        """In-place n_steps of Alg. 1 with the backtracking line search (afsat_step_ls).
        Returns (F, eta, sat_count, is_solution, first_step, converged)."""
        import torch
        self._check_x(x)
        dev = x.device
        F = torch.empty(self.B, dtype=x.dtype, device=dev) if want_F else None
        eta = torch.empty(self.B, dtype=x.dtype, device=dev)
        sat = torch.empty(self.B, dtype=torch.int32, device=dev)
        if state is None:
            sol = torch.empty(self.B, dtype=torch.uint8, device=dev)
            first = torch.empty(self.B, dtype=torch.int32, device=dev)
            conv = torch.empty(self.B, dtype=torch.uint8, device=dev)
            resume = 0
        else:
            sol, first, conv = state
            resume = 1
        hp = None
        if h_any_solved is not None:
            assert h_any_solved.is_pinned() and h_any_solved.dtype == torch.int32 and h_any_solved.numel() >= 2
            hp = h_any_solved.data_ptr()
        rc = self._L.afsat_step_ls(self._h, x.data_ptr(), float(s_max), float(beta), float(c1), float(delta),
                                   int(max_trials), int(n_steps), int(step_base), resume,
                                   F.data_ptr() if F is not None else None, eta.data_ptr(), sat.data_ptr(),
                                   sol.data_ptr(), first.data_ptr(), conv.data_ptr(), hp, _stream_ptr(stream))
        self._raise(rc)
        return F, eta, sat, sol, first, conv

    def restart(self, x, seed, round_, *, keep=None, stream=None):
        """Counter-based uniform re-initialisation of the candidates with keep[b] == 0 (afsat_restart)."""
        self._check_x(x)
        rc = self._L.afsat_restart(self._h, x.data_ptr(), keep.data_ptr() if keep is not None else None,
                                   int(seed), int(round_) & 0xFFFFFFFF, _stream_ptr(stream))
        self._raise(rc)
        return x

    def solve(self, x, eta, steps_per_round, max_rounds, seed, *, stop_at_first=True, want_F=True, stream=None):
        """The restart loop around step (afsat_solve).  Returns (F, sat_count, is_solution, first_step, rounds)."""
        import torch
        self._check_x(x)
        dev = x.device
        F = torch.empty(self.B, dtype=x.dtype, device=dev) if want_F else None
        sat = torch.empty(self.B, dtype=torch.int32, device=dev)
        sol = torch.empty(self.B, dtype=torch.uint8, device=dev)
        first = torch.empty(self.B, dtype=torch.int32, device=dev)
        rounds = C.c_int32(0)
        rc = self._L.afsat_solve(self._h, x.data_ptr(), float(eta), int(steps_per_round), int(max_rounds), int(seed),
                                 1 if stop_at_first else 0, F.data_ptr() if F is not None else None, sat.data_ptr(),
                                 sol.data_ptr(), first.data_ptr(), C.addressof(rounds), _stream_ptr(stream))
        self._raise(rc)
        return F, sat, sol, first, int(rounds.value)

    def step_host(self, h_x, eta, n_steps, *, want_F=True, F_pre=None):
        """End-to-end call on HOST buffers (numpy or pinned torch CPU tensors), synchronous.
        h_x [n, ldb] is updated in place.  Returns (F, sat_count, is_solution, first_step) numpy; F_pre (numpy [B],
        optional) receives F(X(n_steps - 1))."""
        np_dtype = np.float32 if self.dtype == 32 else np.float64
        xp = h_x.data_ptr() if hasattr(h_x, "data_ptr") else h_x.ctypes.data
        assert tuple(h_x.shape) == (self.n, self.ldb)
        F = np.empty(self.B, dtype=np_dtype) if want_F else None
        sat = np.empty(self.B, dtype=np.int32)
        sol = np.empty(self.B, dtype=np.uint8)
        first = np.empty(self.B, dtype=np.int32)
        rc = self._L.afsat_step_host(self._h, xp, float(eta), int(n_steps), _np_ptr(F), _np_ptr(F_pre), sat.ctypes.data,
                                     sol.ctypes.data, first.ctypes.data)
        self._raise(rc)
        return F, sat, sol, first

    def set_profiling(self, on: bool):
        self._raise(self._L.afsat_set_profiling(self._h, 1 if on else 0))

    def profiled_eval_ms(self):
        """(device ms spent in the evaluation kernels, number of their launches) since
        set_profiling(True); synchronises."""
        return self.query(Q_PROFILED_EVAL_NS) * 1e-6, self.query(Q_PROFILED_EVAL_LAUNCHES)

    def query(self, key: int) -> int:
        return int(self._L.afsat_query(self._h, key))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.afsat_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
