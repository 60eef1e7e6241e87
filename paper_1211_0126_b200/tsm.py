"""Thin Python binding over the C-ABI library libtsm.so (include/tsm.h).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the
C ABI.  PyTorch is used for device memory (the workspace, native-layout buffers) and
streams.  There is no CPU fallback: if the library is missing or no CUDA device is
present, construction fails loudly.  Names mirror the C entry points.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtsm.so")

OK, EINVAL, ESTATE, ECUDA, ENOTUNITARY, EBREAKDOWN, ENOCONV = 0, -1, -2, -3, -4, -5, -6
F64, F32, BF16, MIXED = 0, 1, 2, 3
Z4, Z2 = 0, 1
OP_D_EO, OP_D_OE, OP_MHAT, OP_MHAT_DAG, OP_M_FULL = 0, 1, 2, 3, 4
MAX_NRHS = 16
OPS_DERIVATIVE, OPS_ONE_END, OPS_GEN_ONE_END, OPS_MOMENTA = 1, 2, 4, 8
MAX_MOMENTA = 16
PREC = {"f64": F64, "f32": F32, "bf16": BF16, "mixed": MIXED}

EXPORTS = [
    "tsm_create", "tsm_destroy", "tsm_last_error", "tsm_field_bytes", "tsm_workspace_bytes",
    "tsm_set_workspace", "tsm_set_stream", "tsm_set_params", "tsm_set_gauge", "tsm_noise",
    "tsm_pack", "tsm_unpack", "tsm_dslash", "tsm_solve", "tsm_solve_async", "tsm_solve_wait", "tsm_get_solution", "tsm_set_solution",
    "tsm_loops_reset", "tsm_loops_set_momenta", "tsm_loops_add_correction", "tsm_loops_add_lp", "tsm_loops_source",
    "tsm_loops_finalize", "tsm_loops_get_state", "tsm_loops_set_state", "tsm_run_loop_set",
    "tsm_set_hp_precision", "tsm_launch_count", "tsm_profile", "tsm_profile_read", "tsm_stencil_kernel_name",
    "tsm_set_stencil_kernel", "tsm_set_graphs", "tsm_probe_su3_tensor", "tsm_noalloc_scratch_bytes", "tsm_loops_local_noalloc",
]


class SolveInfo(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("status", ctypes.c_int), ("rel_resid_rec", ctypes.c_double),
                ("rel_resid_true", ctypes.c_double), ("secs", ctypes.c_double)]


class TsmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tsm error {code}: {msg}")
        self.code = code


_lib = None


def load_library():
    """dlopen libtsm.so and declare the signatures.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1211_0126_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, dp, i, u64, sz = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_uint64, ctypes.c_size_t
    ip, u32p = ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_uint32)
    lib.tsm_create.argtypes = [ctypes.POINTER(vp), ip, i, i]
    lib.tsm_destroy.argtypes = [vp]
    lib.tsm_last_error.argtypes = [vp]
    lib.tsm_last_error.restype = ctypes.c_char_p
    lib.tsm_field_bytes.argtypes = [vp, i, i]
    lib.tsm_field_bytes.restype = sz
    lib.tsm_workspace_bytes.argtypes = [vp, i, i]
    lib.tsm_workspace_bytes.restype = sz
    lib.tsm_set_workspace.argtypes = [vp, vp, sz, i, i]
    lib.tsm_set_stream.argtypes = [vp, vp]
    lib.tsm_set_params.argtypes = [vp, ctypes.c_double, ctypes.c_double]
    lib.tsm_set_gauge.argtypes = [vp, vp, i, dp]
    lib.tsm_noise.argtypes = [vp, u64, ctypes.c_uint32, i, dp]
    lib.tsm_pack.argtypes = [vp, i, i, dp, vp]
    lib.tsm_unpack.argtypes = [vp, i, i, vp, dp]
    lib.tsm_dslash.argtypes = [vp, i, i, i, vp, vp]
    lib.tsm_solve.argtypes = [vp, u64, u32p, i, i, i, ctypes.c_double, i, i, i, ctypes.POINTER(SolveInfo)]
    lib.tsm_solve_async.argtypes = [vp, u64, u32p, i, i, i, ctypes.c_double, i, i]
    lib.tsm_solve_wait.argtypes = [vp, i, i, ctypes.POINTER(SolveInfo)]
    lib.tsm_get_solution.argtypes = [vp, i, i, dp]
    lib.tsm_set_solution.argtypes = [vp, i, i, dp]
    lib.tsm_loops_reset.argtypes = [vp, i]
    lib.tsm_loops_set_momenta.argtypes = [vp, i, ip]
    lib.tsm_loops_add_correction.argtypes = [vp, i, i]
    lib.tsm_loops_add_lp.argtypes = [vp, i]
    lib.tsm_loops_source.argtypes = [vp, i, i, dp]
    lib.tsm_loops_finalize.argtypes = [vp, dp]
    lib.tsm_loops_get_state.argtypes = [vp, dp, dp, ip, ip]
    lib.tsm_loops_set_state.argtypes = [vp, dp, dp, i, i]
    lib.tsm_run_loop_set.argtypes = [vp, u64, i, i, i, i, ctypes.c_double, i, ctypes.c_double, i, i, i, dp, dp]
    lib.tsm_set_hp_precision.argtypes = [vp, i]
    lib.tsm_launch_count.argtypes = [vp]
    lib.tsm_launch_count.restype = ctypes.c_longlong
    lib.tsm_stencil_kernel_name.argtypes = [vp, i, i]
    lib.tsm_stencil_kernel_name.restype = ctypes.c_char_p
    lib.tsm_set_stencil_kernel.argtypes = [vp, i]
    lib.tsm_noalloc_scratch_bytes.argtypes = []
    lib.tsm_noalloc_scratch_bytes.restype = sz
    lib.tsm_loops_local_noalloc.argtypes = [vp, i, i, vp, u64, u32p, i, vp]
    lib.tsm_probe_su3_tensor.argtypes = [vp, i, i, i, i, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    lib.tsm_set_graphs.argtypes = [vp, i]
    lib.tsm_profile.argtypes = [vp, i]
    lib.tsm_profile_read.argtypes = [vp, i, i, i, dp, ctypes.POINTER(ctypes.c_longlong)]
    _lib = lib
    return lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _host_c128(a, shape) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if a.shape != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {a.shape}")
    return a


class Tsm:
    """One lattice geometry on one GPU; owns the context and the torch workspace tensor."""

    def __init__(self, dims, t_boundary: int = -1, device: int = 0, max_nrhs: int = 1, stream=None, workspace_prec: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1211_0126_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        self.Lt = self.dims[3]
        self.device = device
        self.max_nrhs = max_nrhs
        self.n_ops = 16
        self.hp_precision = MIXED          # the library's default for the HP solves of run_loop_set
        self._h = ctypes.c_void_p()
        rc = self.lib.tsm_create(ctypes.byref(self._h), (ctypes.c_int * 4)(*self.dims), t_boundary, device)
        if rc != OK:
            raise TsmError(rc, "tsm_create failed (extents must be even and >= 4; device must exist)")
        nbytes = self.lib.tsm_workspace_bytes(self._h, max_nrhs, workspace_prec)
        if nbytes == 0:
            raise TsmError(EINVAL, "bad max_nrhs or workspace precision (F64 = everything, F32 = low-precision solves only)")
        self.workspace_prec = workspace_prec
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{device}")
        self._check(self.lib.tsm_set_workspace(self._h, self.workspace.data_ptr(), nbytes, max_nrhs, workspace_prec))
        if stream is not None:
            self.set_stream(stream)

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise TsmError(rc, self.lib.tsm_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.torch.cuda.synchronize(self.device)
            self.lib.tsm_destroy(self._h)
            self._h = ctypes.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        self._check(self.lib.tsm_set_stream(self._h, ctypes.c_void_p(stream.cuda_stream)))

    def launch_count(self) -> int:
        return int(self.lib.tsm_launch_count(self._h))

    def profile(self, enable: bool):
        self._check(self.lib.tsm_profile(self._h, int(enable)))

    def profile_read(self, prec: int, kind: int, nrhs: int = 0):
        """(total ms, launches) recorded for one kernel class since the last read."""
        ms, n = ctypes.c_double(), ctypes.c_longlong()
        self._check(self.lib.tsm_profile_read(self._h, prec, kind, nrhs, ctypes.byref(ms), ctypes.byref(n)))
        return ms.value, n.value

    def field_bytes(self, prec: int, nrhs: int = 1) -> int:
        return int(self.lib.tsm_field_bytes(self._h, prec, nrhs))

    def alloc_field(self, prec: int, nrhs: int = 1, full: bool = False):
        """Native-layout device buffer: single parity, or [parity] full lattice."""
        n = self.field_bytes(prec, nrhs) * (2 if full else 1)
        return self.torch.zeros(n, dtype=self.torch.uint8, device=f"cuda:{self.device}")

    # ------------------------------------------------------------------ the calls of include/tsm.h
    def set_params(self, kappa: float, mu: float):
        self._check(self.lib.tsm_set_params(self._h, kappa, mu))

    def set_hp_precision(self, prec: int):
        """MIXED (default) or F64: how tsm_run_loop_set does its HP solves."""
        self._check(self.lib.tsm_set_hp_precision(self._h, prec))
        self.hp_precision = prec

    def set_stencil_kernel(self, which: int):
        """0 automatic, 1 k_dslash, 2 k_dslash_tile, 3 k_dslash_box, 5 k_dslash_small (tuning / test aid)."""
        self._check(self.lib.tsm_set_stencil_kernel(self._h, which))

    def loops_local_noalloc(self, prec: int, field, seed: int, source_ids, out, kind: int = Z4):
        """tsm_loops_local_noalloc: local loops of the native full-lattice `field` (a torch uint8 tensor, as pack() returns)
        into `out`, a caller-allocated torch float64 tensor of shape [nrhs][16][Lt][2] on the device.  Asynchronous."""
        ids = [int(s) for s in source_ids]
        arr = (ctypes.c_uint32 * len(ids))(*ids)
        self._check(self.lib.tsm_loops_local_noalloc(self._h, prec, len(ids), field.data_ptr(), seed, arr, kind, out.data_ptr()))
        return out

    def probe_su3_tensor(self, variant: int, nsites: int, inner: int, reps: int):
        """(microseconds per launch, max error relative to the largest fp64 reference value) of the per-site
        SU(3) x (3 x 24) product in formulation `variant` (include/tsm.h: tsm_probe_su3_tensor)."""
        us, err = ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.tsm_probe_su3_tensor(self._h, variant, nsites, inner, reps, ctypes.byref(us), ctypes.byref(err)))
        return us.value, err.value

    def set_graphs(self, mode):
        """4 (default): automatic (3 on the smallest lattices, else 1); 1 / True: cached graphs of 4 CG iterations; 2: the CG loop as one graph launch with a device-side
        WHILE node; 3: one cooperative launch of the persistent CG kernel (small lattices); 0 / False: kernel by kernel."""
        self._check(self.lib.tsm_set_graphs(self._h, int(mode)))

    def hp_precision_name(self) -> str:
        return "mixed" if self.hp_precision == MIXED else "fp64"

    def stencil_kernel_name(self, prec: int, nrhs: int) -> str:
        """Name of the stencil kernel the library launches for this precision and batch size."""
        return self.lib.tsm_stencil_kernel_name(self._h, prec, nrhs).decode()

    def set_gauge(self, links, reconstruct: int = 18) -> float:
        """links: host complex128 [4][V][3][3], or a pinned torch tensor viewing the same bytes."""
        dev = ctypes.c_double(-1.0)
        if isinstance(links, np.ndarray):
            a = _host_c128(links, (4, self.V, 3, 3))
            ptr = a.ctypes.data
        else:   # torch CPU tensor (pinned for the e2e path), float64 [4][V][3][3][2]
            if links.device.type != "cpu" or links.dtype != self.torch.float64 or links.numel() != 4 * self.V * 18:
                raise ValueError("links tensor must be CPU float64 with 4*V*18 elements")
            a = links.contiguous()
            ptr = a.data_ptr()
        self._check(self.lib.tsm_set_gauge(self._h, ctypes.c_void_p(ptr), reconstruct, ctypes.byref(dev)))
        return dev.value

    def noise(self, seed: int, source_id: int, kind: int = Z4) -> np.ndarray:
        out = np.empty((self.V, 4, 3), dtype=np.complex128)
        self._check(self.lib.tsm_noise(self._h, seed, source_id, kind, _dptr(out)))
        return out

    def pack(self, prec: int, host_lex, out=None):
        a = np.ascontiguousarray(host_lex, dtype=np.complex128)
        if a.ndim == 3:
            a = a[None]
        nrhs = a.shape[0]
        a = _host_c128(a, (nrhs, self.V, 4, 3))
        buf = self.alloc_field(prec, nrhs, full=True) if out is None else out
        self._check(self.lib.tsm_pack(self._h, prec, nrhs, _dptr(a), buf.data_ptr()))
        return buf

    def unpack(self, prec: int, nrhs: int, buf) -> np.ndarray:
        out = np.empty((nrhs, self.V, 4, 3), dtype=np.complex128)
        self._check(self.lib.tsm_unpack(self._h, prec, nrhs, buf.data_ptr(), _dptr(out)))
        return out

    def dslash(self, op: int, prec: int, nrhs: int, dev_in, dev_out):
        self._check(self.lib.tsm_dslash(self._h, op, prec, nrhs, dev_in.data_ptr(), dev_out.data_ptr()))

    def solve(self, seed: int, source_ids, prec: int, tol: float, max_iter: int, slot: int = 0,
              kind: int = Z4, want_true_resid: bool = False):
        """Returns (rc, [dict per source]); rc is OK, EBREAKDOWN or ENOCONV (solutions are kept)."""
        ids = [int(s) for s in source_ids]
        n = len(ids)
        arr = (ctypes.c_uint32 * n)(*ids)
        info = (SolveInfo * n)()
        rc = self.lib.tsm_solve(self._h, seed, arr, n, kind, prec, tol, max_iter, slot, int(want_true_resid), info)
        self._check(rc, allow=(EBREAKDOWN, ENOCONV))
        return rc, [dict(iters=x.iters, status=x.status, rel_resid_rec=x.rel_resid_rec,
                         rel_resid_true=x.rel_resid_true, secs=x.secs) for x in info]

    def solve_async(self, seed: int, source_ids, prec: int, tol: float, max_iter: int, slot: int = 0, kind: int = Z4):
        """Enqueue a solve without waiting for it (tsm_solve_async); solve_wait(slot) reports on it later."""
        ids = [int(s) for s in source_ids]
        arr = (ctypes.c_uint32 * len(ids))(*ids)
        self._pending_n = getattr(self, "_pending_n", {})
        self._pending_n[slot] = len(ids)
        self._check(self.lib.tsm_solve_async(self._h, seed, arr, len(ids), kind, prec, tol, max_iter, slot))

    def solve_wait(self, slot: int = 0, want_true_resid: bool = False):
        """(rc, [dict per source]) of the solve last enqueued into `slot`, as solve() would have returned it."""
        n = getattr(self, "_pending_n", {}).get(slot, self.max_nrhs)
        info = (SolveInfo * n)()
        rc = self.lib.tsm_solve_wait(self._h, slot, int(want_true_resid), info)
        self._check(rc, allow=(EBREAKDOWN, ENOCONV))
        return rc, [dict(iters=x.iters, status=x.status, rel_resid_rec=x.rel_resid_rec,
                         rel_resid_true=x.rel_resid_true, secs=x.secs) for x in info]

    def get_solution(self, slot: int, rhs: int) -> np.ndarray:
        out = np.empty((self.V, 4, 3), dtype=np.complex128)
        self._check(self.lib.tsm_get_solution(self._h, slot, rhs, _dptr(out)))
        return out

    def set_solution(self, slot: int, rhs: int, s):
        a = _host_c128(s, (self.V, 4, 3))
        self._check(self.lib.tsm_set_solution(self._h, slot, rhs, _dptr(a)))

    @staticmethod
    def _ops(with_derivative: bool, one_end: bool, gen_one_end: bool = False) -> int:
        return ((OPS_DERIVATIVE if with_derivative else 0) | (OPS_ONE_END if one_end else 0)
                | (OPS_GEN_ONE_END if gen_one_end else 0))

    def loops_reset(self, with_derivative: bool = False, one_end: bool = False, gen_one_end: bool = False, momenta=None):
        """n_ops = 16 local [+ 64 derivative] [+ 16 one-end (Eq. 2.5)] [+ 16 generalised one-end (Eq. 2.6)]
        [+ 16 per momentum of `momenta` ([nmom][3] integers, p_i = 2 pi n_i / L_i)]."""
        ops = self._ops(with_derivative, one_end, gen_one_end)
        nmom = 0
        if momenta is not None:
            mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
            nmom = mom.shape[0]
            self._check(self.lib.tsm_loops_set_momenta(self._h, nmom, mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
            ops |= OPS_MOMENTA
        self.n_ops = 16 + (64 if with_derivative else 0) + (16 if one_end else 0) + (16 if gen_one_end else 0) + 16 * nmom
        self._check(self.lib.tsm_loops_reset(self._h, ops))

    def loops_add_correction(self, slot_hp: int, slot_lp: int):
        self._check(self.lib.tsm_loops_add_correction(self._h, slot_hp, slot_lp))

    def loops_add_lp(self, slot_lp: int):
        self._check(self.lib.tsm_loops_add_lp(self._h, slot_lp))

    def loops_source(self, slot: int, rhs: int) -> np.ndarray:
        out = np.empty((self.n_ops, self.Lt), dtype=np.complex128)
        self._check(self.lib.tsm_loops_source(self._h, slot, rhs, _dptr(out)))
        return out

    def loops_finalize(self) -> np.ndarray:
        out = np.empty((self.n_ops, self.Lt), dtype=np.complex128)
        self._check(self.lib.tsm_loops_finalize(self._h, _dptr(out)))
        return out

    def loops_get_state(self):
        corr = np.empty((self.n_ops, self.Lt), dtype=np.complex128)
        lp = np.empty((self.n_ops, self.Lt), dtype=np.complex128)
        n_hp, n_lp = ctypes.c_int(), ctypes.c_int()
        self._check(self.lib.tsm_loops_get_state(self._h, _dptr(corr), _dptr(lp), ctypes.byref(n_hp), ctypes.byref(n_lp)))
        return corr, lp, n_hp.value, n_lp.value

    def loops_set_state(self, corr, lp, n_hp: int, n_lp: int):
        corr = _host_c128(corr, (self.n_ops, self.Lt))
        lp = _host_c128(lp, (self.n_ops, self.Lt))
        self._check(self.lib.tsm_loops_set_state(self._h, _dptr(corr), _dptr(lp), n_hp, n_lp))

    def run_loop_set(self, seed: int, n_hp: int, n_lp: int, lp_prec: int, lp_tol: float, lp_iters: int,
                     hp_tol: float = 1e-10, hp_max_iter: int = 5000, nrhs: int = 1,
                     with_derivative: bool = False, kind: int = Z4, one_end: bool = False, gen_one_end: bool = False,
                     momenta=None):
        """Eq. 2.4 for one configuration.  Returns (loops [n_ops][Lt], device seconds, rc)."""
        ops = self._ops(with_derivative, one_end, gen_one_end)
        nmom = 0
        if momenta is not None:
            mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
            nmom = mom.shape[0]
            self._check(self.lib.tsm_loops_set_momenta(self._h, nmom, mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
            ops |= OPS_MOMENTA
        self.n_ops = 16 + (64 if with_derivative else 0) + (16 if one_end else 0) + (16 if gen_one_end else 0) + 16 * nmom
        out = np.empty((self.n_ops, self.Lt), dtype=np.complex128)
        secs = ctypes.c_double(0.0)
        rc = self.lib.tsm_run_loop_set(self._h, seed, kind, n_hp, n_lp, lp_prec, lp_tol, lp_iters, hp_tol,
                                       hp_max_iter, nrhs, ops, _dptr(out), ctypes.byref(secs))
        self._check(rc, allow=(EBREAKDOWN, ENOCONV))
        return out, secs.value, rc
