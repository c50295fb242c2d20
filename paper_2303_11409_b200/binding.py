"""Thin ctypes binding of libu1mps.so (include/u1mps.h).  Argument marshalling only: every step of
the two-site update runs in the CUDA kernels of the library.  PyTorch is used for device memory
(the arena) and the stream.  There is no CPU fallback: if the library is missing, or no CUDA
device is present, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libu1mps.so")

EXPORTS = [
    "u1mps_strerror", "u1mps_version", "u1mps_workspace_bytes", "u1mps_create", "u1mps_destroy",
    "u1mps_set_product_state", "u1mps_apply_two_site_gate", "u1mps_stage_theta", "u1mps_stage_svd",
    "u1mps_truncate", "u1mps_apply_and_truncate", "u1mps_apply_gate_column", "u1mps_norm2", "u1mps_log_norm",
    "u1mps_expect_n", "u1mps_expect_n_all", "u1mps_bond_entropy", "u1mps_bond_entropy_all", "u1mps_bond_info",
    "u1mps_bond_dims", "u1mps_last_stats", "u1mps_export_bond", "u1mps_export_site", "u1mps_import_bond",
    "u1mps_import_site", "u1mps_set_log_norm", "u1mps_staged_info", "u1mps_export_staged_theta",
    "u1mps_export_staged_svd", "u1mps_launch_count", "u1mps_profile_enable", "u1mps_profile_read",
    "u1mps_stage_name", "u1mps_svd_trace", "u1mps_clear_status", "u1mps_expect_n_full_bytes", "u1mps_expect_n_full",
    "u1mps_expect_nn_full_bytes", "u1mps_expect_nn_full", "u1mps_expect_n_all_static",
    "u1mps_sample_fock_bytes", "u1mps_sample_fock",
]
NSTAGE = 8

ENOCONV = -6
ETOOBIG = -7
STATIC_SITES_MAX = 1024   # U1MPS_STATIC_SITES_MAX


class U1MPSError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libu1mps error {code}: {msg}")
        self.code = code


_lib = None


def load_library() -> C.CDLL:
    """dlopen libu1mps.so (built in-tree by paper_2303_11409_b200.build).  Fails loudly if missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not found: run `python -m paper_2303_11409_b200.build` "
                                "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32p, dp = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_double)
    lib.u1mps_strerror.restype = C.c_char_p
    lib.u1mps_strerror.argtypes = [C.c_int]
    lib.u1mps_version.restype = C.c_char_p
    lib.u1mps_workspace_bytes.restype = C.c_size_t
    lib.u1mps_workspace_bytes.argtypes = [C.c_int] * 4
    lib.u1mps_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, vp, C.c_size_t, vp]
    lib.u1mps_destroy.argtypes = [vp]
    lib.u1mps_set_product_state.argtypes = [vp, i32p]
    lib.u1mps_apply_two_site_gate.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.u1mps_stage_theta.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.u1mps_stage_svd.argtypes = [vp]
    lib.u1mps_truncate.argtypes = [vp, C.c_int, C.c_int, C.c_double]
    lib.u1mps_apply_and_truncate.argtypes = [vp, C.c_int, vp, C.c_int, C.c_int, C.c_double]
    lib.u1mps_apply_gate_column.argtypes = [vp, i32p, C.c_int, vp, C.c_int, C.c_int, C.c_double]
    lib.u1mps_norm2.argtypes = [vp, dp]
    lib.u1mps_log_norm.argtypes = [vp, dp]
    lib.u1mps_expect_n.argtypes = [vp, C.c_int, dp]
    lib.u1mps_expect_n_all.argtypes = [vp, dp]
    lib.u1mps_bond_entropy.argtypes = [vp, C.c_int, dp]
    lib.u1mps_bond_entropy_all.argtypes = [vp, dp]
    lib.u1mps_bond_info.argtypes = [vp, C.c_int, i32p, i32p, i32p, C.c_int]
    lib.u1mps_bond_dims.argtypes = [vp, i32p]
    lib.u1mps_last_stats.argtypes = [vp, dp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.u1mps_export_bond.argtypes = [vp, C.c_int, dp, C.c_int]
    lib.u1mps_export_site.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_size_t]
    lib.u1mps_import_bond.argtypes = [vp, C.c_int, C.c_int, i32p, i32p, dp]
    lib.u1mps_import_site.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_size_t]
    lib.u1mps_set_log_norm.argtypes = [vp, C.c_double, C.c_double]
    lib.u1mps_staged_info.argtypes = [vp, i32p, i32p, i32p, i32p, C.c_int]
    lib.u1mps_export_staged_theta.argtypes = [vp, C.c_int, vp, C.c_size_t]
    lib.u1mps_export_staged_svd.argtypes = [vp, C.c_int, vp, dp, vp]
    lib.u1mps_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
    lib.u1mps_profile_enable.argtypes = [vp, C.c_int]
    lib.u1mps_profile_read.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
    lib.u1mps_svd_trace.argtypes = [vp, C.POINTER(C.c_longlong), C.c_int]
    lib.u1mps_clear_status.argtypes = [vp]
    lib.u1mps_expect_n_full_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    lib.u1mps_expect_n_full.argtypes = [vp, dp, vp, C.c_size_t]
    lib.u1mps_expect_nn_full_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    lib.u1mps_expect_nn_full.argtypes = [vp, C.c_int, C.c_int, dp, vp, C.c_size_t]
    lib.u1mps_expect_n_all_static.argtypes = [vp, vp]
    lib.u1mps_sample_fock_bytes.argtypes = [vp, C.c_int, C.POINTER(C.c_size_t)]
    lib.u1mps_sample_fock.argtypes = [vp, C.c_int, dp, i32p, dp, vp, C.c_size_t]
    lib.u1mps_stage_name.restype = C.c_char_p
    lib.u1mps_stage_name.argtypes = [C.c_int]
    for name in EXPORTS:
        if name not in ("u1mps_strerror", "u1mps_version", "u1mps_workspace_bytes", "u1mps_stage_name"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a: np.ndarray, typ):
    return a.ctypes.data_as(typ)


class U1MPS:
    """Handle of one U(1) MPS on the current CUDA device.  Method names follow the C ABI."""

    def __init__(self, M: int, d: int, N: int, chi: int, arena_bytes: Optional[int] = None, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libu1mps needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.M, self.d, self.N, self.chi = M, d, N, chi
        need = self.lib.u1mps_workspace_bytes(M, d, N, chi)
        if need == 0:
            raise U1MPSError(-1, "invalid dimensions")
        nbytes = max(need, int(arena_bytes or 0))
        self.arena = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.h = C.c_void_p()
        self._ck(self.lib.u1mps_create(C.byref(self.h), M, d, N, chi, C.c_void_p(self.arena.data_ptr()), nbytes,
                                       C.c_void_p(self.stream.cuda_stream)))

    # ------------------------------------------------------------------ helpers
    def _ck(self, code: int, allow=()):
        if code != 0 and code not in allow:
            raise U1MPSError(code, self.lib.u1mps_strerror(code).decode())
        return code

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self.lib.u1mps_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _gate_arg(U):
        """Returns (pointer, on_device, keepalive) for a numpy array (host) or a torch CUDA tensor (device)."""
        if isinstance(U, np.ndarray):
            a = np.ascontiguousarray(U, dtype=np.complex128)
            return C.c_void_p(a.ctypes.data), 0, a
        import torch
        if isinstance(U, torch.Tensor):
            assert U.dtype == torch.complex128 and U.is_contiguous()
            if U.is_cuda:
                return C.c_void_p(U.data_ptr()), 1, U
            return C.c_void_p(U.data_ptr()), 0, U
        raise TypeError("gate must be a numpy array or a torch tensor")

    # ------------------------------------------------------------------ state
    def set_product_state(self, occ: Sequence[int]):
        a = _i32(occ)
        if a.shape != (self.M,):
            raise U1MPSError(-1, "occ must have length M")
        self._ck(self.lib.u1mps_set_product_state(self.h, _ptr(a, C.POINTER(C.c_int32))))

    # ------------------------------------------------------------------ the update
    def apply_two_site_gate(self, i: int, U):
        p, dev, keep = self._gate_arg(U)
        self._ck(self.lib.u1mps_apply_two_site_gate(self.h, i, p, dev))

    def stage_theta(self, i: int, U):
        p, dev, keep = self._gate_arg(U)
        self._ck(self.lib.u1mps_stage_theta(self.h, i, p, dev))

    def stage_svd(self):
        self._ck(self.lib.u1mps_stage_svd(self.h))

    def truncate(self, i: int, chi: Optional[int] = None, cutoff: float = 1e-12):
        self._ck(self.lib.u1mps_truncate(self.h, i, self.chi if chi is None else chi, cutoff))

    def apply_and_truncate(self, i: int, U, chi: Optional[int] = None, cutoff: float = 1e-12):
        p, dev, keep = self._gate_arg(U)
        self._ck(self.lib.u1mps_apply_and_truncate(self.h, i, p, dev, self.chi if chi is None else chi, cutoff))

    def apply_gate_column(self, sites, U, chi: Optional[int] = None, cutoff: float = 1e-12):
        s = _i32(sites)
        p, dev, keep = self._gate_arg(U)
        self._ck(self.lib.u1mps_apply_gate_column(self.h, _ptr(s, C.POINTER(C.c_int32)), len(s), p, dev,
                                                  self.chi if chi is None else chi, cutoff))

    # ------------------------------------------------------------------ readouts
    def norm2(self, allow_nonconverged: bool = False) -> float:
        """Raises U1MPSError(ENOCONV) if any SVD since the last clear_status() hit the sweep limit (unless allowed)."""
        v = C.c_double()
        self._ck(self.lib.u1mps_norm2(self.h, C.byref(v)), allow=(ENOCONV,) if allow_nonconverged else ())
        return v.value

    def log_norm(self, allow_nonconverged: bool = False) -> float:
        v = C.c_double()
        self._ck(self.lib.u1mps_log_norm(self.h, C.byref(v)), allow=(ENOCONV,) if allow_nonconverged else ())
        return v.value

    def clear_status(self):
        self._ck(self.lib.u1mps_clear_status(self.h))

    def expect_n(self, site: int) -> float:
        v = C.c_double()
        self._ck(self.lib.u1mps_expect_n(self.h, site, C.byref(v)))
        return v.value

    def expect_n_all(self) -> np.ndarray:
        out = np.zeros(self.M)
        self._ck(self.lib.u1mps_expect_n_all(self.h, _ptr(out, C.POINTER(C.c_double))))
        return out

    def expect_n_all_static(self, out_dev) -> None:
        """u1mps_expect_n_all on the library's static scratch: no allocation, no synchronisation.  out_dev: a CUDA
        float64 tensor of M elements that the caller owns; it is valid once the handle's stream has got there."""
        if not (out_dev.is_cuda and out_dev.dtype.is_floating_point and out_dev.element_size() == 8
                and out_dev.is_contiguous() and out_dev.numel() >= self.M):
            raise U1MPSError(-1, "out_dev must be a contiguous CUDA float64 tensor of at least M elements")
        self._ck(self.lib.u1mps_expect_n_all_static(self.h, C.c_void_p(out_dev.data_ptr())))

    def sample_fock(self, u) -> Tuple[np.ndarray, np.ndarray]:
        """Fock patterns drawn from |<n|psi>|^2 / <psi|psi>; u: [B, M] uniform numbers in [0, 1) (the caller's random
        numbers).  Returns (pattern int32 [B, M], logp [B])."""
        import torch
        u = np.ascontiguousarray(u, dtype=np.float64)
        if u.ndim != 2 or u.shape[1] != self.M:
            raise U1MPSError(-1, "u must be [n_samples, M]")
        B = u.shape[0]
        nbytes = C.c_size_t()
        self._ck(self.lib.u1mps_sample_fock_bytes(self.h, B, C.byref(nbytes)))
        scratch = torch.empty(max(nbytes.value, 256), dtype=torch.uint8, device="cuda")
        pat = np.zeros((B, self.M), dtype=np.int32)
        logp = np.zeros(B)
        self._ck(self.lib.u1mps_sample_fock(self.h, B, _ptr(u, C.POINTER(C.c_double)), _ptr(pat, C.POINTER(C.c_int32)),
                                            _ptr(logp, C.POINTER(C.c_double)), C.c_void_p(scratch.data_ptr()), nbytes.value))
        return pat, logp

    def expect_n_full(self) -> np.ndarray:
        """<psi|n_k|psi> / <psi|psi> with explicit environments (exact also after truncation); scratch from torch."""
        import torch
        nbytes = C.c_size_t()
        self._ck(self.lib.u1mps_expect_n_full_bytes(self.h, C.byref(nbytes)))
        scratch = torch.empty(max(nbytes.value, 256), dtype=torch.uint8, device="cuda")
        out = np.zeros(self.M)
        self._ck(self.lib.u1mps_expect_n_full(self.h, _ptr(out, C.POINTER(C.c_double)), C.c_void_p(scratch.data_ptr()), nbytes.value))
        return out

    def expect_nn_full(self, j: int, k: int) -> float:
        """<psi|n_j n_k|psi> / <psi|psi> with explicit environments."""
        import torch
        nbytes = C.c_size_t()
        self._ck(self.lib.u1mps_expect_nn_full_bytes(self.h, C.byref(nbytes)))
        scratch = torch.empty(max(nbytes.value, 256), dtype=torch.uint8, device="cuda")
        v = C.c_double()
        self._ck(self.lib.u1mps_expect_nn_full(self.h, j, k, C.byref(v), C.c_void_p(scratch.data_ptr()), nbytes.value))
        return v.value

    def bond_entropy(self, bond: int) -> float:
        v = C.c_double()
        self._ck(self.lib.u1mps_bond_entropy(self.h, bond, C.byref(v)))
        return v.value

    def bond_entropy_all(self) -> np.ndarray:
        out = np.zeros(self.M + 1)
        self._ck(self.lib.u1mps_bond_entropy_all(self.h, _ptr(out, C.POINTER(C.c_double))))
        return out

    def bond_info(self, bond: int) -> List[Tuple[int, int]]:
        cap = self.N + 1
        ch, cn = np.zeros(cap, np.int32), np.zeros(cap, np.int32)
        n = C.c_int32()
        self._ck(self.lib.u1mps_bond_info(self.h, bond, C.byref(n), _ptr(ch, C.POINTER(C.c_int32)),
                                          _ptr(cn, C.POINTER(C.c_int32)), cap))
        return [(int(ch[k]), int(cn[k])) for k in range(n.value)]

    def bond_dims(self) -> np.ndarray:
        out = np.zeros(self.M + 1, np.int32)
        self._ck(self.lib.u1mps_bond_dims(self.h, _ptr(out, C.POINTER(C.c_int32))))
        return out

    def last_stats(self) -> Dict[str, float]:
        dw, kept, sw = C.c_double(), C.c_int(), C.c_int()
        code = self._ck(self.lib.u1mps_last_stats(self.h, C.byref(dw), C.byref(kept), C.byref(sw)), allow=(ENOCONV,))
        return {"discarded": dw.value, "kept": kept.value, "sweeps": sw.value, "converged": code == 0}

    def profile_enable(self, on: bool = True):
        self._ck(self.lib.u1mps_profile_enable(self.h, 1 if on else 0))

    def profile_read(self) -> Dict[str, Tuple[float, int]]:
        """{stage name: (summed device ms, launches)} since the last read."""
        ms = np.zeros(NSTAGE)
        n = np.zeros(NSTAGE, np.int64)
        self._ck(self.lib.u1mps_profile_read(self.h, _ptr(ms, C.POINTER(C.c_double)), _ptr(n, C.POINTER(C.c_longlong))))
        return {self.lib.u1mps_stage_name(s).decode(): (float(ms[s]), int(n[s])) for s in range(NSTAGE)}

    def svd_trace(self) -> Dict[str, np.ndarray]:
        """Per-sweep trace of the last a3 launch: ms per sweep, rotated pair items, inner EVD sweeps, active sectors."""
        ms_ = 30
        raw = np.zeros(4 * ms_ + 1, np.int64)
        self._ck(self.lib.u1mps_svd_trace(self.h, _ptr(raw, C.POINTER(C.c_longlong)), len(raw)))
        t = np.concatenate([[raw[0]], raw[1:1 + ms_]])
        n = int(np.count_nonzero(raw[1:1 + ms_]))
        return {"sweep_ms": np.diff(t[:n + 1]) * 1e-6, "rotated_items": raw[1 + ms_:1 + ms_ + n],
                "inner_sweeps": raw[1 + 2 * ms_:1 + 2 * ms_ + n], "active_sectors": raw[1 + 3 * ms_:1 + 3 * ms_ + n]}

    def launch_count(self) -> int:
        v = C.c_longlong()
        self._ck(self.lib.u1mps_launch_count(self.h, C.byref(v)))
        return v.value

    # ------------------------------------------------------------------ export / import
    def export_bond(self, bond: int) -> Dict[int, np.ndarray]:
        info = self.bond_info(bond)
        D = sum(n for _, n in info)
        lam = np.zeros(D)
        self._ck(self.lib.u1mps_export_bond(self.h, bond, _ptr(lam, C.POINTER(C.c_double)), D))
        out, off = {}, 0
        for c, n in info:
            out[c] = lam[off:off + n].copy()
            off += n
        return out

    def export_site(self, site: int) -> Dict[Tuple[int, int], np.ndarray]:
        left, right = dict(self.bond_info(site)), dict(self.bond_info(site + 1))
        out = {}
        for cl, nl in left.items():
            for i in range(self.d):
                cr = cl - i
                if cr in right:
                    blk = np.zeros((nl, right[cr]), dtype=np.complex128)
                    self._ck(self.lib.u1mps_export_site(self.h, site, cl, cr, C.c_void_p(blk.ctypes.data), blk.nbytes))
                    out[(cl, cr)] = blk
        return out

    def import_bond(self, bond: int, lam_by_charge: Dict[int, np.ndarray]):
        ch = sorted(lam_by_charge)
        cn = [len(lam_by_charge[c]) for c in ch]
        lam = np.ascontiguousarray(np.concatenate([np.asarray(lam_by_charge[c], dtype=np.float64) for c in ch]))
        a, b = _i32(ch), _i32(cn)
        self._ck(self.lib.u1mps_import_bond(self.h, bond, len(ch), _ptr(a, C.POINTER(C.c_int32)),
                                            _ptr(b, C.POINTER(C.c_int32)), _ptr(lam, C.POINTER(C.c_double))))

    def import_site(self, site: int, blocks: Dict[Tuple[int, int], np.ndarray]):
        for (cl, cr), blk in blocks.items():
            a = np.ascontiguousarray(blk, dtype=np.complex128)
            self._ck(self.lib.u1mps_import_site(self.h, site, cl, cr, C.c_void_p(a.ctypes.data), a.nbytes))

    def import_state(self, lam: Sequence[Dict[int, np.ndarray]], gam: Sequence[Dict[Tuple[int, int], np.ndarray]],
                     log_norm: float = 0.0, discarded: float = 0.0):
        """Load a whole state given as plain dictionaries (bonds first, then sites)."""
        for k in range(self.M + 1):
            self.import_bond(k, lam[k])
        for s in range(self.M):
            self.import_site(s, gam[s])
        self._ck(self.lib.u1mps_set_log_norm(self.h, log_norm, discarded))

    # ------------------------------------------------------------------ staged read-back
    def staged_info(self) -> List[Tuple[int, int, int]]:
        cap = self.N + 1
        ch, r, q = np.zeros(cap, np.int32), np.zeros(cap, np.int32), np.zeros(cap, np.int32)
        n = C.c_int32()
        ip = C.POINTER(C.c_int32)
        self._ck(self.lib.u1mps_staged_info(self.h, C.byref(n), _ptr(ch, ip), _ptr(r, ip), _ptr(q, ip), cap),
                 allow=(ENOCONV,))
        return [(int(ch[k]), int(r[k]), int(q[k])) for k in range(n.value)]

    def export_staged_theta(self, c: int, rows: int, cols: int) -> np.ndarray:
        out = np.zeros((rows, cols), dtype=np.complex128)
        self._ck(self.lib.u1mps_export_staged_theta(self.h, c, C.c_void_p(out.ctypes.data), out.nbytes))
        return out

    def export_staged_svd(self, c: int, rows: int, cols: int):
        r = min(rows, cols)
        V = np.zeros((rows, r), dtype=np.complex128)
        S = np.zeros(r)
        W = np.zeros((r, cols), dtype=np.complex128)
        self._ck(self.lib.u1mps_export_staged_svd(self.h, c, C.c_void_p(V.ctypes.data), _ptr(S, C.POINTER(C.c_double)),
                                                  C.c_void_p(W.ctypes.data)), allow=(ENOCONV,))
        return V, S, W
