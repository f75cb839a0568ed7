"""Thin Python binding of libtt.so (include/tt.h): argument marshalling only.

Same names as the C ABI.  PyTorch supplies device memory and streams; every step of the hot path
runs inside the library's CUDA kernels.  There is no CPU fallback: importing works anywhere (so
that CPU-only tests can check the exported symbols), but creating a context without the built
library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes
import os
from pathlib import Path

import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = Path(os.environ["TT_LIB_PATH"]) if os.environ.get("TT_LIB_PATH") else _HERE / "libtt.so"   # override: A/B builds

TT_OK = 0
TT_F64, TT_F32 = 0, 1
TT_HESS_EQ4, TT_HESS_FILTER, TT_HESS_PSD2, TT_HESS_PSDPROJ, TT_HESS_EXACT = 0, 1, 2, 3, 4
TT_STATIC_MAX_PAIRS = 1 << 24   # tt_energy_static (include/tt.h)
TT_FLAG_FORCE_GENERAL_ROWS = 1
TT_FLAG_VALIDATE_INDICES = 2
TT_FLAG_NO_STATE_CHECK = 4

EXPORTS = ["tt_create", "tt_destroy", "tt_energy", "tt_energy_static", "tt_hess_symbolic", "tt_energy_grad_hess", "tt_hess_vec",
           "tt_energy_grad_hess_host", "tt_hess_pattern", "tt_broad_phase", "tt_broad_phase_pairs", "tt_broad_phase_copy", "tt_bsr_device", "tt_bsr_spmv", "tt_block_jacobi", "tt_pcg_solve", "tt_newton_step", "tt_untangle", "tt_membrane_build", "tt_membrane_energy_grad", "tt_membrane_hess_vec", "tt_stats", "tt_kernel_ms", "tt_kernel_ms_mean", "tt_probe_peaks", "tt_probe_gather", "tt_status_string", "tt_last_error"]


class TTOptions(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int32), ("hess_mode", ctypes.c_int32), ("tc_scale", ctypes.c_double),
                ("device", ctypes.c_int32), ("flags", ctypes.c_int32)]


class TTProblem(ctypes.Structure):
    _fields_ = [("pos", ctypes.c_void_p), ("n_verts", ctypes.c_int64), ("tris", ctypes.c_void_p),
                ("n_tris", ctypes.c_int64), ("pairs", ctypes.c_void_p), ("n_pairs", ctypes.c_int64)]


class TTPcgOptions(ctypes.Structure):
    _fields_ = [("max_iter", ctypes.c_int32), ("check_every", ctypes.c_int32), ("rtol", ctypes.c_double),
                ("shift", ctypes.c_double)]


class TTNewtonOptions(ctypes.Structure):
    _fields_ = [("mu", ctypes.c_double), ("armijo_c1", ctypes.c_double), ("max_backtrack", ctypes.c_int32),
                ("matrix_free", ctypes.c_int32), ("pcg", TTPcgOptions), ("membrane", ctypes.c_int32),
                ("reserved", ctypes.c_int32)]


class TTNewtonReport(ctypes.Structure):
    _fields_ = [("energy0", ctypes.c_double), ("energy1", ctypes.c_double), ("grad_norm", ctypes.c_double),
                ("gd", ctypes.c_double), ("alpha", ctypes.c_double), ("pcg_relres", ctypes.c_double),
                ("n_pairs", ctypes.c_int64), ("n_active", ctypes.c_int64), ("nnzb", ctypes.c_int64),
                ("pcg_iters", ctypes.c_int32), ("backtracks", ctypes.c_int32), ("accepted", ctypes.c_int32),
                ("reserved", ctypes.c_int32), ("energy_membrane", ctypes.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class TTError(RuntimeError):
    def __init__(self, status, name, msg):
        super().__init__("%s (%d): %s" % (name, status, msg))
        self.status = status


_lib = None


def load_library():
    """dlopen libtt.so and declare the C signatures.  Raises if the library was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError("libtt.so is missing (%s): run `python -m paper_2606_06511_b200.build` "
                           "or __graft_entry__.build(); there is no CPU fallback" % LIB_PATH)
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, i64 = ctypes.c_void_p, ctypes.c_int64
    lib.tt_create.argtypes = [ctypes.POINTER(TTOptions), ctypes.POINTER(vp)]
    lib.tt_create.restype = ctypes.c_int
    lib.tt_destroy.argtypes = [vp]
    lib.tt_destroy.restype = None
    lib.tt_energy.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, vp, vp, vp, vp]
    lib.tt_energy.restype = ctypes.c_int
    lib.tt_energy_static.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, vp]
    lib.tt_energy_static.restype = ctypes.c_int
    lib.tt_hess_symbolic.argtypes = [vp, ctypes.POINTER(TTProblem), ctypes.POINTER(i64), ctypes.POINTER(i64), vp]
    lib.tt_hess_symbolic.restype = ctypes.c_int
    lib.tt_energy_grad_hess.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, vp, vp, vp, i64, vp]
    lib.tt_energy_grad_hess.restype = ctypes.c_int
    lib.tt_hess_vec.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, vp]
    lib.tt_hess_vec.restype = ctypes.c_int
    lib.tt_energy_grad_hess_host.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, ctypes.POINTER(i64),
                                             ctypes.POINTER(i64), vp, vp, vp, i64, vp, vp, vp]
    lib.tt_energy_grad_hess_host.restype = ctypes.c_int
    lib.tt_broad_phase.argtypes = [vp, vp, i64, vp, i64, ctypes.c_double, ctypes.POINTER(i64), vp]
    lib.tt_broad_phase.restype = ctypes.c_int
    lib.tt_broad_phase_pairs.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i64)]
    lib.tt_broad_phase_pairs.restype = ctypes.c_int
    lib.tt_broad_phase_copy.argtypes = [vp, vp, i64, vp]
    lib.tt_broad_phase_copy.restype = ctypes.c_int
    lib.tt_hess_pattern.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64)]
    lib.tt_hess_pattern.restype = ctypes.c_int
    lib.tt_bsr_device.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64)]
    lib.tt_bsr_device.restype = ctypes.c_int
    lib.tt_bsr_spmv.argtypes = [vp, i64, vp, vp, vp, ctypes.c_double, vp, vp, vp]
    lib.tt_bsr_spmv.restype = ctypes.c_int
    lib.tt_block_jacobi.argtypes = [vp, i64, vp, vp, vp, ctypes.c_double, vp, vp]
    lib.tt_block_jacobi.restype = ctypes.c_int
    lib.tt_pcg_solve.argtypes = [vp, ctypes.POINTER(TTProblem), vp, vp, vp, vp, vp, vp, ctypes.POINTER(TTPcgOptions),
                                 ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_double), vp]
    lib.tt_pcg_solve.restype = ctypes.c_int
    lib.tt_newton_step.argtypes = [vp, vp, i64, vp, i64, vp, i64, ctypes.POINTER(TTNewtonOptions),
                                   ctypes.POINTER(TTNewtonReport), vp]
    lib.tt_newton_step.restype = ctypes.c_int
    lib.tt_untangle.argtypes = [vp, vp, i64, vp, i64, ctypes.c_double, ctypes.c_int32, ctypes.POINTER(TTNewtonOptions),
                                ctypes.POINTER(TTNewtonReport), ctypes.POINTER(ctypes.c_int32), vp]
    lib.tt_untangle.restype = ctypes.c_int
    lib.tt_membrane_build.argtypes = [vp, vp, i64, vp, i64, ctypes.c_double, vp]
    lib.tt_membrane_build.restype = ctypes.c_int
    lib.tt_membrane_energy_grad.argtypes = [vp, vp, vp, vp, vp]
    lib.tt_membrane_energy_grad.restype = ctypes.c_int
    lib.tt_membrane_hess_vec.argtypes = [vp, vp, vp, vp, vp]
    lib.tt_membrane_hess_vec.restype = ctypes.c_int
    lib.tt_stats.argtypes = [vp, ctypes.POINTER(i64), ctypes.c_int32]
    lib.tt_stats.restype = ctypes.c_int
    lib.tt_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.c_int32]
    lib.tt_kernel_ms.restype = ctypes.c_int
    lib.tt_kernel_ms_mean.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int32), ctypes.c_int32,
                                      ctypes.c_int32]
    lib.tt_kernel_ms_mean.restype = ctypes.c_int
    lib.tt_probe_peaks.argtypes = [ctypes.c_int32, ctypes.POINTER(ctypes.c_double)]
    lib.tt_probe_peaks.restype = ctypes.c_int
    lib.tt_probe_gather.argtypes = [ctypes.c_int32, ctypes.POINTER(ctypes.c_double)]
    lib.tt_probe_gather.restype = ctypes.c_int
    lib.tt_status_string.argtypes = [ctypes.c_int]
    lib.tt_status_string.restype = ctypes.c_char_p
    lib.tt_last_error.argtypes = [vp]
    lib.tt_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _ptr(t):
    """Device pointer of a tensor; raw addresses (int / c_void_p, e.g. from tt_hess_pattern_ptrs) pass through."""
    if t is None or isinstance(t, ctypes.c_void_p):
        return t
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    return ctypes.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class Context:
    """Owns a tt_ctx.  dtype: torch.float64 or torch.float32."""

    def __init__(self, dtype=torch.float64, hess_mode=TT_HESS_FILTER, tc_scale=1.0, device=0, flags=0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_06511_b200 needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.dtype = dtype
        self.device = torch.device("cuda", device)
        opt = TTOptions(TT_F64 if dtype == torch.float64 else TT_F32, int(hess_mode), float(tc_scale), int(device), int(flags))
        h = ctypes.c_void_p()
        st = self.lib.tt_create(ctypes.byref(opt), ctypes.byref(h))
        if st != TT_OK:
            raise TTError(st, self.lib.tt_status_string(st).decode(), "tt_create failed")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.tt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != TT_OK:
            raise TTError(st, self.lib.tt_status_string(st).decode(), self.lib.tt_last_error(self.h).decode())

    def problem(self, pos, tris, pairs):
        """Builds a tt_problem view of device tensors (kept alive by the returned tuple)."""
        assert pos.is_cuda and tris.is_cuda and pairs.is_cuda
        assert pos.dtype == self.dtype and tris.dtype == torch.int32 and pairs.dtype == torch.int32
        assert pos.is_contiguous() and tris.is_contiguous() and pairs.is_contiguous()
        pb = TTProblem(pos.data_ptr(), pos.shape[0], tris.data_ptr(), tris.shape[0], pairs.data_ptr(), pairs.shape[0])
        return pb, (pos, tris, pairs)

    # ---- tt_energy ----
    def tt_energy(self, prob, energy_sum, energy_per_pair=None, active_mask=None, tc=None, n_active=None, stream=None):
        self._check(self.lib.tt_energy(self.h, ctypes.byref(prob[0]), _ptr(energy_sum), _ptr(energy_per_pair),
                                       _ptr(active_mask), _ptr(tc), _ptr(n_active), _stream_ptr(stream)))

    def tt_energy_static(self, prob, energy_sum, n_active=None, stream=None):
        """tt_energy's total (and active count) with the scratch in the library's static device array: no allocation,
        no synchronisation; at most TT_STATIC_MAX_PAIRS candidates."""
        self._check(self.lib.tt_energy_static(self.h, ctypes.byref(prob[0]), _ptr(energy_sum), _ptr(n_active),
                                              _stream_ptr(stream)))

    # ---- tt_hess_symbolic ----
    def tt_hess_symbolic(self, prob, stream=None):
        nnzb, na = ctypes.c_int64(0), ctypes.c_int64(0)
        self._check(self.lib.tt_hess_symbolic(self.h, ctypes.byref(prob[0]), ctypes.byref(nnzb), ctypes.byref(na),
                                              _stream_ptr(stream)))
        return nnzb.value, na.value

    # ---- tt_energy_grad_hess ----
    def tt_energy_grad_hess(self, prob, energy_sum, grad=None, bsr_rowptr=None, bsr_colind=None, bsr_vals=None,
                            nnzb_capacity=0, stream=None):
        self._check(self.lib.tt_energy_grad_hess(self.h, ctypes.byref(prob[0]), _ptr(energy_sum), _ptr(grad),
                                                 _ptr(bsr_rowptr), _ptr(bsr_colind), _ptr(bsr_vals),
                                                 int(nnzb_capacity), _stream_ptr(stream)))

    # ---- tt_hess_pattern ----
    def tt_hess_pattern_ptrs(self):
        """(rowptr address, colind address, nnzb) of the ctx-owned pattern -- re-read after every tt_hess_symbolic (the
        workspace may have been re-allocated)."""
        rp, ci, n = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_int64(0)
        self._check(self.lib.tt_hess_pattern(self.h, ctypes.byref(rp), ctypes.byref(ci), ctypes.byref(n)))
        return rp.value, ci.value, int(n.value)

    def tt_hess_pattern(self, n_verts):
        """Zero-copy int32 tensor views (rowptr [nV+1], colind [nnzb]) of the ctx-owned pattern of the last
        tt_hess_symbolic; valid until the next symbolic / host call.  Passing them to tt_energy_grad_hess skips its
        pattern copy."""
        rp, ci, n = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_int64(0)
        self._check(self.lib.tt_hess_pattern(self.h, ctypes.byref(rp), ctypes.byref(ci), ctypes.byref(n)))

        class _View:
            def __init__(self, ptr, count):
                self.__cuda_array_interface__ = dict(shape=(count,), typestr="<i4", data=(ptr, False), version=2)

        rowptr = torch.as_tensor(_View(rp.value, int(n_verts) + 1), device=self.device)
        colind = torch.as_tensor(_View(ci.value, max(int(n.value), 1)), device=self.device)
        return rowptr, colind, int(n.value)

    # ---- tt_hess_vec ----
    def tt_hess_vec(self, prob, p, y, stream=None):
        self._check(self.lib.tt_hess_vec(self.h, ctypes.byref(prob[0]), _ptr(p), _ptr(y), _stream_ptr(stream)))

    # ---- tt_energy_grad_hess_host ----
    def tt_energy_grad_hess_host(self, pos_h, tris_h, pairs_h, energy_h, grad_h=None, rowptr_h=None, colind_h=None,
                                 vals_h=None, nnzb_capacity=0, p_h=None, y_h=None, stream=None):
        """All tensors are HOST tensors (pinned recommended).  Returns (nnzb, n_active)."""
        for t in (pos_h, tris_h, pairs_h, energy_h):
            assert not t.is_cuda and t.is_contiguous()
        pb = TTProblem(pos_h.data_ptr(), pos_h.shape[0], tris_h.data_ptr(), tris_h.shape[0], pairs_h.data_ptr(),
                       pairs_h.shape[0])
        nnzb, na = ctypes.c_int64(0), ctypes.c_int64(0)
        self._check(self.lib.tt_energy_grad_hess_host(self.h, ctypes.byref(pb), _ptr(energy_h), _ptr(grad_h),
                                                      ctypes.byref(nnzb), ctypes.byref(na), _ptr(rowptr_h),
                                                      _ptr(colind_h), _ptr(vals_h), int(nnzb_capacity),
                                                      _ptr(p_h), _ptr(y_h), _stream_ptr(stream)))
        return nnzb.value, na.value

    def tt_broad_phase(self, pos, tris, inflate=0.0, stream=None):
        """Candidate pairs of (pos, tris): returns a new int32 [P,2] device tensor (tt_broad_phase +
        tt_broad_phase_copy)."""
        n = ctypes.c_int64(0)
        sp = _stream_ptr(stream)
        assert pos.dtype == self.dtype and tris.dtype == torch.int32 and pos.is_contiguous() and tris.is_contiguous()
        self._check(self.lib.tt_broad_phase(self.h, _ptr(pos), pos.shape[0], _ptr(tris), tris.shape[0], float(inflate),
                                            ctypes.byref(n), sp))
        out = torch.empty((int(n.value), 2), dtype=torch.int32, device=pos.device)
        self._check(self.lib.tt_broad_phase_copy(self.h, _ptr(out) if n.value else None, int(n.value), sp))
        return out

    # ---- the consumer: BSR product, block-Jacobi, PCG ----
    def tt_bsr_spmv(self, rowptr, colind, vals, x, y, shift=0.0, stream=None):
        self._check(self.lib.tt_bsr_spmv(self.h, x.shape[0], _ptr(rowptr), _ptr(colind), _ptr(vals), float(shift), _ptr(x),
                                         _ptr(y), _stream_ptr(stream)))

    def tt_block_jacobi(self, rowptr, colind, vals, minv, shift=0.0, stream=None):
        self._check(self.lib.tt_block_jacobi(self.h, minv.shape[0], _ptr(rowptr), _ptr(colind), _ptr(vals), float(shift),
                                             _ptr(minv), _stream_ptr(stream)))

    def tt_pcg_solve(self, prob, b, x, rowptr=None, colind=None, vals=None, minv=None, max_iter=50, rtol=0.0, shift=0.0,
                     check_every=0, want_stats=True, stream=None):
        """vals given: assembled (BSR) back end; vals None: matrix-free (tt_hess_vec).  Returns (iters, relres)
        (synchronises) or None with want_stats=False (fully asynchronous when rtol == 0)."""
        opt = TTPcgOptions(int(max_iter), int(check_every), float(rtol), float(shift))
        it, rr = ctypes.c_int32(0), ctypes.c_double(0.0)
        self._check(self.lib.tt_pcg_solve(self.h, ctypes.byref(prob[0]), _ptr(rowptr), _ptr(colind), _ptr(vals), _ptr(minv),
                                          _ptr(b), _ptr(x), ctypes.byref(opt), ctypes.byref(it) if want_stats else None,
                                          ctypes.byref(rr) if want_stats else None, _stream_ptr(stream)))
        return (it.value, rr.value) if want_stats else None

    @staticmethod
    def _newton_options(mu, c1, max_backtrack, matrix_free, pcg_iter, pcg_rtol, membrane=False):
        return TTNewtonOptions(float(mu), float(c1), int(max_backtrack), 1 if matrix_free else 0,
                               TTPcgOptions(int(pcg_iter), 0, float(pcg_rtol), 0.0), 1 if membrane else 0, 0)

    def tt_membrane_build(self, rest_pos, tris, stiffness, stream=None):
        """Adjacency + rest lengths of the edge-spring membrane of `tris` (owned by the context)."""
        assert rest_pos.is_cuda and rest_pos.dtype == self.dtype and rest_pos.is_contiguous()
        assert tris.is_cuda and tris.dtype == torch.int32 and tris.is_contiguous()
        self._check(self.lib.tt_membrane_build(self.h, _ptr(rest_pos), rest_pos.shape[0], _ptr(tris), tris.shape[0],
                                               float(stiffness), _stream_ptr(stream)))

    def tt_membrane_energy_grad(self, pos, want_grad=True, stream=None):
        """E_m (a 1-element fp64 device tensor) and its gradient ([nV,3] dtype, or None)."""
        assert pos.is_cuda and pos.dtype == self.dtype and pos.is_contiguous()
        e = torch.empty(1, dtype=torch.float64, device=pos.device)
        g = torch.empty_like(pos) if want_grad else None
        self._check(self.lib.tt_membrane_energy_grad(self.h, _ptr(pos), _ptr(e), _ptr(g) if want_grad else None,
                                                     _stream_ptr(stream)))
        return e, g

    def tt_membrane_hess_vec(self, pos, p, stream=None):
        assert pos.is_cuda and pos.dtype == self.dtype and pos.is_contiguous()
        assert p.is_cuda and p.dtype == self.dtype and p.is_contiguous() and p.shape == pos.shape
        y = torch.empty_like(p)
        self._check(self.lib.tt_membrane_hess_vec(self.h, _ptr(pos), _ptr(p), _ptr(y), _stream_ptr(stream)))
        return y

    def tt_newton_step(self, pos, tris, pairs, mu=1e-3, c1=1e-4, max_backtrack=20, matrix_free=False, pcg_iter=20,
                       pcg_rtol=0.0, membrane=False, stream=None):
        """One damped inexact-Newton step; `pos` is updated IN PLACE.  Returns the report as a dict."""
        assert pos.is_cuda and pos.dtype == self.dtype and pos.is_contiguous()
        opt = self._newton_options(mu, c1, max_backtrack, matrix_free, pcg_iter, pcg_rtol, membrane)
        rep = TTNewtonReport()
        self._check(self.lib.tt_newton_step(self.h, _ptr(pos), pos.shape[0], _ptr(tris), tris.shape[0], _ptr(pairs),
                                            pairs.shape[0], ctypes.byref(opt), ctypes.byref(rep), _stream_ptr(stream)))
        return rep.as_dict()

    def tt_untangle(self, pos, tris, inflate=0.0, max_steps=20, mu=1e-3, c1=1e-4, max_backtrack=20, matrix_free=False,
                    pcg_iter=20, pcg_rtol=0.0, membrane=False, stream=None):
        """Broad phase + Newton step until nothing intersects; `pos` is updated IN PLACE.  Returns the list of reports."""
        assert pos.is_cuda and pos.dtype == self.dtype and pos.is_contiguous()
        opt = self._newton_options(mu, c1, max_backtrack, matrix_free, pcg_iter, pcg_rtol, membrane)
        hist = (TTNewtonReport * max(int(max_steps), 1))()
        n = ctypes.c_int32(0)
        self._check(self.lib.tt_untangle(self.h, _ptr(pos), pos.shape[0], _ptr(tris), tris.shape[0], float(inflate),
                                         int(max_steps), ctypes.byref(opt), hist, ctypes.byref(n), _stream_ptr(stream)))
        return [hist[i].as_dict() for i in range(n.value)]

    def tt_kernel_ms(self):
        arr = (ctypes.c_float * 3)()
        self._check(self.lib.tt_kernel_ms(self.h, arr, 3))
        return dict(classify=float(arr[0]), assemble=float(arr[1]), hess_vec=float(arr[2]))

    def tt_kernel_ms_mean(self, reset=False):
        """Mean duration of the launches recorded since the last reset: (dict of ms, dict of launch counts)."""
        arr = (ctypes.c_float * 3)()
        cnt = (ctypes.c_int32 * 3)()
        self._check(self.lib.tt_kernel_ms_mean(self.h, arr, cnt, 3, 1 if reset else 0))
        names = ("classify", "assemble", "hess_vec")
        return {k: float(arr[i]) for i, k in enumerate(names)}, {k: int(cnt[i]) for i, k in enumerate(names)}

    def tt_stats(self):
        arr = (ctypes.c_int64 * 13)()
        self._check(self.lib.tt_stats(self.h, arr, 13))
        keys = ["n_active", "n_directed", "n_touched_tris", "blocks_direct", "blocks_merged", "merge_records", "nnzb",
                "launches", "n_slots", "split_triangles", "parts", "long_rounds", "rounds"]
        return dict(zip(keys, [int(v) for v in arr]))


def tt_probe_peaks(device=0):
    """Measured DFMA / FFMA rate of `device` in TFLOP/s (diagnostic)."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_06511_b200 needs a CUDA device (no CPU fallback)")
    lib = load_library()
    arr = (ctypes.c_double * 2)()
    st = lib.tt_probe_peaks(int(device), arr)
    if st != TT_OK:
        raise TTError(st, lib.tt_status_string(st).decode(), "tt_probe_peaks failed")
    return dict(fp64_tflops=float(arr[0]), fp32_tflops=float(arr[1]))


def tt_probe_gather(device=0):
    """Useful GB/s of random 24-byte / 72-byte gathers from a 144 MB array (diagnostic)."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_06511_b200 needs a CUDA device (no CPU fallback)")
    lib = load_library()
    arr = (ctypes.c_double * 2)()
    st = lib.tt_probe_gather(int(device), arr)
    if st != TT_OK:
        raise TTError(st, lib.tt_status_string(st).decode(), "tt_probe_gather failed")
    return dict(vertex_gbs=float(arr[0]), triangle_gbs=float(arr[1]))


def assemble(ctx: Context, pos, tris, pairs, want_hess=True, stream=None):
    """Convenience: symbolic + allocate + numeric.  Returns dict of device tensors."""
    prob = ctx.problem(pos, tris, pairs)
    nnzb, n_active = ctx.tt_hess_symbolic(prob, stream)
    dev, dt = pos.device, ctx.dtype
    energy = torch.zeros(1, dtype=dt, device=dev)
    grad = torch.empty((pos.shape[0], 3), dtype=dt, device=dev)
    out = dict(energy=energy, grad=grad, nnzb=nnzb, n_active=n_active, prob=prob)
    if want_hess:
        rowptr = torch.empty(pos.shape[0] + 1, dtype=torch.int32, device=dev)
        colind = torch.empty(max(nnzb, 1), dtype=torch.int32, device=dev)
        vals = torch.empty((max(nnzb, 1), 3, 3), dtype=dt, device=dev)
        ctx.tt_energy_grad_hess(prob, energy, grad, rowptr, colind, vals, max(nnzb, 1), stream)
        out.update(rowptr=rowptr, colind=colind[:nnzb], vals=vals[:nnzb])
    else:
        ctx.tt_energy_grad_hess(prob, energy, grad, None, None, None, 0, stream)
    return out
