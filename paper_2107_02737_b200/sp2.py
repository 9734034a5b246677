"""Thin Python binding of the C ABI in include/sp2.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of ``libsp2_b200.so``; PyTorch is used here only
to own device memory (the workspace and the matrices) and to name the current stream.  There is
no CPU fallback: importing this module raises if the library has not been built
(``python -m paper_2107_02737_b200.build``), and every call raises ``Sp2Error`` on a non-OK status
other than "not converged".

Names follow include/sp2.h: ``workspace_bytes``, ``Sp2Handle.density`` (sp2_density),
``.response`` (sp2_response), ``.density_host`` / ``.response_host`` (host-buffer twins),
``.sequence_begin/step/end`` (sp2_sequence_*).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libsp2_b200.so")

SP2_OK = 0
SP2_ERR_INVALID_ARG = 1
SP2_ERR_WORKSPACE = 2
SP2_ERR_CUDA = 3
SP2_ERR_ARCH = 4
SP2_ERR_NONFINITE = 5
SP2_ERR_DEGENERATE = 6
SP2_WARN_NOT_CONVERGED = 7
SP2_ERR_BOUNDS = 8
SP2_ERR_TOO_LARGE = 9

SP2_F32, SP2_F64 = 0, 1
SP2_WITH_RESPONSE, SP2_WITH_HOST_STAGING, SP2_WITH_REFINEMENT = 1, 2, 4
SP2_MAX_BATCH = 8


def SP2_WITH_BATCH(nb: int) -> int:
    return (int(nb) & 15) << 8

SP2_ENGINE_TCGEN05, SP2_ENGINE_SIMT_DEBUG = 0, 1

EXPORTS = [
    "sp2_workspace_bytes", "sp2_create", "sp2_destroy", "sp2_set_options", "sp2_get_options",
    "sp2_density", "sp2_response", "sp2_response_batch", "sp2_density_host", "sp2_response_host",
    "sp2_sequence_begin", "sp2_sequence_step", "sp2_sequence_end", "sp2_congruence",
    "sp2_status_string", "sp2_last_cuda_error", "sp2_launch_count",
    "sp2_density_noalloc", "sp2_noalloc_max_n", "sp2_noalloc_scratch_bytes",
    "sp2_debug_history", "sp2_debug_plane", "sp2_debug_schedule", "sp2_debug_layout",
]


class Sp2Options(C.Structure):
    _fields_ = [
        ("max_layers", C.c_int), ("user_bounds", C.c_int),
        ("eps_min", C.c_double), ("eps_max", C.c_double),
        ("engine", C.c_int), ("forced_layers", C.c_int),
        ("forced_signs", C.c_ulonglong), ("cta_group", C.c_int),
        ("lanczos_steps", C.c_int), ("refine_layers", C.c_int), ("seg_kb", C.c_int), ("lo_bits", C.c_int), ("no_recentre", C.c_int),
        ("persistent", C.c_int), ("max_ctas", C.c_int), ("power_squarings", C.c_int), ("lockstep", C.c_int),
    ]


class Sp2Result(C.Structure):
    _fields_ = [
        ("status", C.c_int), ("layers", C.c_int),
        ("sign_mask", C.c_ulonglong * 2),
        ("stop_reason", C.c_int), ("reserved", C.c_int),
        ("tr_d", C.c_double), ("tr_dh", C.c_double), ("tr_d1", C.c_double),
        ("idem_est", C.c_double), ("eps_min", C.c_double), ("eps_max", C.c_double),
        ("gpu_ms", C.c_float), ("layers_ms", C.c_float), ("kernel_launches", C.c_int), ("bounds_fallback", C.c_int),
    ]

    def as_dict(self):
        signs = "".join(
            "+" if (self.sign_mask[n >> 6] >> (n & 63)) & 1 else "-" for n in range(self.layers))
        return dict(status=self.status, layers=self.layers, signs=signs, stop_reason=self.stop_reason,
                    refine_layers=self.reserved, tr_d=self.tr_d, tr_dh=self.tr_dh, tr_d1=self.tr_d1, idem_est=self.idem_est,
                    eps_min=self.eps_min, eps_max=self.eps_max, gpu_ms=self.gpu_ms, layers_ms=self.layers_ms,
                    kernel_launches=self.kernel_launches, bounds_fallback=self.bounds_fallback)


class Sp2Error(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"sp2 status {status}: {msg}")
        self.status = status


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2107_02737_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i, d, l, sz = C.c_void_p, C.c_int, C.c_double, C.c_long, C.c_size_t
    lib.sp2_workspace_bytes.restype = sz
    lib.sp2_workspace_bytes.argtypes = [i, i]
    lib.sp2_create.restype = i
    lib.sp2_create.argtypes = [C.POINTER(vp), i, i, vp, sz]
    lib.sp2_destroy.restype = i
    lib.sp2_destroy.argtypes = [vp]
    lib.sp2_set_options.restype = i
    lib.sp2_set_options.argtypes = [vp, C.POINTER(Sp2Options)]
    lib.sp2_get_options.restype = i
    lib.sp2_get_options.argtypes = [vp, C.POINTER(Sp2Options)]
    dens = [vp, vp, i, l, i, i, d, vp, i, l, C.POINTER(Sp2Result), vp]
    resp = [vp, vp, vp, i, l, i, i, d, vp, vp, i, l, C.POINTER(Sp2Result), vp]
    for name, args in (("sp2_density", dens), ("sp2_density_host", dens),
                       ("sp2_response", resp), ("sp2_response_host", resp)):
        f = getattr(lib, name)
        f.restype = i
        f.argtypes = args
    lib.sp2_response_batch.restype = i
    lib.sp2_response_batch.argtypes = [vp, vp, C.POINTER(vp), i, i, l, i, i, d, vp, C.POINTER(vp), i, l, C.POINTER(d),
                                       C.POINTER(Sp2Result), vp]
    lib.sp2_sequence_begin.restype = i
    lib.sp2_sequence_begin.argtypes = [vp, i, i, d, i, vp]
    lib.sp2_sequence_step.restype = i
    lib.sp2_sequence_step.argtypes = [vp, vp, i, l, vp, i, l]
    lib.sp2_sequence_end.restype = i
    lib.sp2_sequence_end.argtypes = [vp, C.POINTER(Sp2Result), C.POINTER(i)]
    lib.sp2_congruence.restype = i
    lib.sp2_congruence.argtypes = [vp, vp, vp, i, l, i, i, vp, i, l, vp]
    lib.sp2_density_noalloc.restype = i
    lib.sp2_density_noalloc.argtypes = [vp, i, l, i, i, d, vp, i, l, vp, C.POINTER(Sp2Result), vp]
    lib.sp2_noalloc_max_n.restype = i
    lib.sp2_noalloc_max_n.argtypes = []
    lib.sp2_noalloc_scratch_bytes.restype = sz
    lib.sp2_noalloc_scratch_bytes.argtypes = []
    lib.sp2_status_string.restype = C.c_char_p
    lib.sp2_status_string.argtypes = [i]
    lib.sp2_last_cuda_error.restype = i
    lib.sp2_last_cuda_error.argtypes = [vp]
    lib.sp2_launch_count.restype = C.c_ulonglong
    lib.sp2_launch_count.argtypes = [vp]
    lib.sp2_debug_history.restype = i
    lib.sp2_debug_history.argtypes = [vp, C.POINTER(d), C.POINTER(d), i]
    lib.sp2_debug_plane.restype = i
    lib.sp2_debug_plane.argtypes = [vp, i, C.POINTER(sz), C.POINTER(l), C.POINTER(i), C.POINTER(d)]
    lib.sp2_debug_layout.restype = i
    lib.sp2_debug_layout.argtypes = [vp, i, C.c_char_p, C.POINTER(sz), C.POINTER(sz), C.POINTER(sz)]
    lib.sp2_debug_schedule.restype = i
    lib.sp2_debug_schedule.argtypes = [i, i, i, i, C.POINTER(i), i, C.POINTER(i)]
    return lib


lib = _load()


def debug_schedule(n_tiles: int, with_response: bool, segs_per_pass: int, n_clusters: int):
    """Host-only: work lists of the layer kernel -> list (per cluster) of dicts."""
    cap = (1 + int(with_response)) * n_tiles * 2 + 4 * n_clusters + 16   # with_response: bool or perturbation count
    buf = (C.c_int * (8 * cap))()
    begin = (C.c_int * (n_clusters + 1))()
    cnt = lib.sp2_debug_schedule(n_tiles, int(with_response), segs_per_pass, n_clusters, buf, cap, begin)
    if cnt < 0 or cnt > cap:
        raise ValueError("bad schedule arguments")
    keys = ("unit", "seg0", "seg1", "kind", "slot", "nparts", "flag_id")
    items = [dict(zip(keys, buf[8 * k:8 * k + 7])) for k in range(cnt)]
    return [items[begin[c]:begin[c + 1]] for c in range(n_clusters)]


def status_string(status: int) -> str:
    return lib.sp2_status_string(int(status)).decode()


def workspace_bytes(n_max: int, flags: int = 0) -> int:
    return int(lib.sp2_workspace_bytes(int(n_max), int(flags)))


def noalloc_max_n() -> int:
    return int(lib.sp2_noalloc_max_n())


def noalloc_scratch_bytes() -> int:
    return int(lib.sp2_noalloc_scratch_bytes())


def density_noalloc(H, n_occ: int, out, tol: float = 0.0, d_result=None, blocking: bool = True):
    """sp2_density_noalloc: H (CUDA tensor, N <= noalloc_max_n()) -> `out` (CUDA tensor the CALLER allocated) with no
    handle and no workspace; scratch is the library's static device array.  Runs on H's device and torch's current
    stream there.  blocking=False only enqueues (pass d_result, a CUDA uint8 tensor of >= 96 bytes, to get the status)."""
    import torch

    n = H.shape[0]
    for t in (H, out):
        if not t.is_cuda or t.dim() != 2 or t.shape[0] != n or t.shape[1] != n or t.stride(1) != 1:
            raise ValueError("expected N x N CUDA tensors with unit column stride")
    if out.device != H.device:
        raise ValueError("H and out must be on the same device")
    r = Sp2Result()
    dres = C.c_void_p(d_result.data_ptr()) if d_result is not None else None
    with torch.cuda.device(H.device):
        stream = C.c_void_p(torch.cuda.current_stream(H.device).cuda_stream)
        st = lib.sp2_density_noalloc(C.c_void_p(H.data_ptr()), _dtype_code(H), H.stride(0), n, int(n_occ), float(tol),
                                     C.c_void_p(out.data_ptr()), _dtype_code(out), out.stride(0), dres,
                                     C.byref(r) if blocking else None, stream)
    if st not in (SP2_OK, SP2_WARN_NOT_CONVERGED):
        raise Sp2Error(st, status_string(st))
    return out, (r.as_dict() if blocking else None)


def _dtype_code(t):
    import torch

    if t.dtype == torch.float32:
        return SP2_F32
    if t.dtype == torch.float64:
        return SP2_F64
    raise TypeError("matrices must be float32 or float64")


def _np_dtype_code(a):
    if a.dtype == np.float32:
        return SP2_F32
    if a.dtype == np.float64:
        return SP2_F64
    raise TypeError("matrices must be float32 or float64")


class Sp2Handle:
    """sp2_create / sp2_destroy over a torch-owned workspace on the current CUDA device."""

    GUARD = 4096   # bytes either side of the workspace when a sentinel is asked for (tests)

    def __init__(self, n_max: int, response: bool = False, host_staging: bool = False, device=None,
                 refinement: bool = False, batch: int = 0, sentinel: int | None = None):
        """sentinel (tests only): fill the workspace and a guard band either side of it with this byte BEFORE
        sp2_create, so that ``debug_layout`` / ``check_canary`` can tell which bytes the library ever wrote."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("sp2-b200 needs a CUDA device (sm_100); there is no CPU fallback")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.flags = ((SP2_WITH_RESPONSE if response else 0) | (SP2_WITH_HOST_STAGING if host_staging else 0)
                      | (SP2_WITH_REFINEMENT if refinement else 0) | (SP2_WITH_BATCH(batch) if batch else 0))
        self.n_max = int(n_max)
        nbytes = workspace_bytes(self.n_max, self.flags)
        self.sentinel = sentinel
        guard = self.GUARD if sentinel is not None else 0
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 1024 + 2 * guard, dtype=torch.uint8, device=self.device)
            if sentinel is not None:
                self.workspace.fill_(int(sentinel))
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + guard + 1023) // 1024 * 1024
            self._ws_off = self._ws_ptr - base
            self._ws_bytes = nbytes
            h = C.c_void_p()
            st = lib.sp2_create(C.byref(h), self.n_max, self.flags, C.c_void_p(self._ws_ptr), nbytes)
        if st != SP2_OK:
            raise Sp2Error(st, status_string(st))
        self._h = h

    # ------------------------------------------------------------------ plumbing
    def close(self):
        if getattr(self, "_h", None):
            lib.sp2_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        import torch

        return C.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    def _raise(self, st):
        if st not in (SP2_OK, SP2_WARN_NOT_CONVERGED):
            extra = ""
            if st == SP2_ERR_CUDA:
                extra = f" (cuda error {lib.sp2_last_cuda_error(self._h)})"
            raise Sp2Error(st, status_string(st) + extra)

    def set_options(self, **kw):
        """Fields of sp2_options_t (include/sp2.h) by name: max_layers, user_bounds=(eps_min, eps_max) | None, engine,
        forced_layers, forced_signs, cta_group, seg_kb, lo_bits, refine_layers, lanczos_steps, persistent, max_ctas,
        power_squarings, lockstep, ...  Keywords change the named fields and keep the others; no keyword restores the
        defaults."""
        if not kw:
            self._raise(lib.sp2_set_options(self._h, None))
            return
        o = Sp2Options()
        self._raise(lib.sp2_get_options(self._h, C.byref(o)))
        for k, v in kw.items():
            if k == "user_bounds":
                if v is None:
                    o.user_bounds = 0
                else:
                    o.user_bounds, o.eps_min, o.eps_max = 1, float(v[0]), float(v[1])
            elif k == "forced_signs" and isinstance(v, str):
                o.forced_signs = sum(1 << n for n, ch in enumerate(v) if ch == "+")
                o.forced_layers = len(v)
            else:
                setattr(o, k, v)
        self._raise(lib.sp2_set_options(self._h, C.byref(o)))

    @property
    def launch_count(self) -> int:
        return int(lib.sp2_launch_count(self._h))

    # ------------------------------------------------------------------ device-pointer calls
    def _check_dev(self, t, n):
        if not t.is_cuda or t.dim() != 2 or t.shape[0] < n or t.shape[1] < n or t.stride(1) != 1:
            raise ValueError("expected a CUDA row-major 2-D tensor of at least N x N")

    def density(self, H, n_occ: int, tol: float = 0.0, out=None, out_dtype=None):
        """sp2_density: H (N x N CUDA tensor, f32/f64) -> (D, result dict)."""
        import torch

        n = H.shape[0]
        self._check_dev(H, n)
        if out is None:
            out = torch.empty((n, n), dtype=out_dtype or H.dtype, device=H.device)
        self._check_dev(out, n)
        r = Sp2Result()
        st = lib.sp2_density(self._h, C.c_void_p(H.data_ptr()), _dtype_code(H), H.stride(0), n, int(n_occ), float(tol),
                             C.c_void_p(out.data_ptr()), _dtype_code(out), out.stride(0), C.byref(r), self._stream())
        self._raise(st)
        return out, r.as_dict()

    def response(self, H, H1, n_occ: int, tol: float = 0.0, out=None, out1=None, out_dtype=None):
        """sp2_response: (H, H1) -> (D, D1, result dict)."""
        import torch

        n = H.shape[0]
        self._check_dev(H, n)
        self._check_dev(H1, n)
        if H1.dtype != H.dtype or H1.stride(0) != H.stride(0):
            raise ValueError("H1 must have the dtype and pitch of H")
        if out is None:
            out = torch.empty((n, n), dtype=out_dtype or H.dtype, device=H.device)
        if out1 is None:
            out1 = torch.empty_like(out)
        if out1.dtype != out.dtype or out1.stride(0) != out.stride(0):
            raise ValueError("D1 must have the dtype and pitch of D")
        r = Sp2Result()
        st = lib.sp2_response(self._h, C.c_void_p(H.data_ptr()), C.c_void_p(H1.data_ptr()), _dtype_code(H), H.stride(0),
                              n, int(n_occ), float(tol), C.c_void_p(out.data_ptr()), C.c_void_p(out1.data_ptr()),
                              _dtype_code(out), out.stride(0), C.byref(r), self._stream())
        self._raise(st)
        return out, out1, r.as_dict()

    def response_batch(self, H, H1s, n_occ: int, tol: float = 0.0, out=None, out1s=None, out_dtype=None):
        """sp2_response_batch: (H, [H1_b]) -> (D, [D1_b], [tr D1_b], result dict); one stack of layers for all b."""
        import torch

        n = H.shape[0]
        nb = len(H1s)
        self._check_dev(H, n)
        for H1 in H1s:
            self._check_dev(H1, n)
            if H1.dtype != H.dtype or H1.stride(0) != H.stride(0):
                raise ValueError("every H1 must have the dtype and pitch of H")
        if out is None:
            out = torch.empty((n, n), dtype=out_dtype or H.dtype, device=H.device)
        if out1s is None:
            out1s = [torch.empty_like(out) for _ in range(nb)]
        for o in out1s:
            if o.dtype != out.dtype or o.stride(0) != out.stride(0):
                raise ValueError("every D1 must have the dtype and pitch of D")
        pin = (C.c_void_p * max(nb, 1))(*[H1.data_ptr() for H1 in H1s])
        pout = (C.c_void_p * max(nb, 1))(*[o.data_ptr() for o in out1s])
        tr = (C.c_double * SP2_MAX_BATCH)()
        r = Sp2Result()
        st = lib.sp2_response_batch(self._h, C.c_void_p(H.data_ptr()), pin, nb, _dtype_code(H), H.stride(0), n, int(n_occ),
                                    float(tol), C.c_void_p(out.data_ptr()), pout, _dtype_code(out), out.stride(0), tr,
                                    C.byref(r), self._stream())
        self._raise(st)
        return out, list(out1s), [tr[b] for b in range(nb)], r.as_dict()

    # ------------------------------------------------------------------ host-buffer calls
    @staticmethod
    def _host_ptr(a):
        """numpy array or CPU torch tensor (pinned or not) -> (pointer, dtype code, pitch, keepalive)."""
        if isinstance(a, np.ndarray):
            if a.ndim != 2 or a.strides[1] != a.itemsize:
                raise ValueError("expected a row-major 2-D array")
            return a.ctypes.data, _np_dtype_code(a), a.strides[0] // a.itemsize, a
        if a.is_cuda or a.dim() != 2 or a.stride(1) != 1:
            raise ValueError("expected a CPU row-major 2-D tensor")
        return a.data_ptr(), _dtype_code(a), a.stride(0), a

    def density_host(self, H, n_occ: int, out, tol: float = 0.0):
        """sp2_density_host: host H -> host `out` (both numpy arrays or CPU tensors); copies inside the call."""
        n = H.shape[0]
        ph, dh, lh, _k1 = self._host_ptr(H)
        po, do, lo, _k2 = self._host_ptr(out)
        r = Sp2Result()
        st = lib.sp2_density_host(self._h, C.c_void_p(ph), dh, lh, n, int(n_occ), float(tol), C.c_void_p(po), do, lo,
                                  C.byref(r), self._stream())
        self._raise(st)
        return out, r.as_dict()

    def response_host(self, H, H1, n_occ: int, out, out1, tol: float = 0.0):
        n = H.shape[0]
        ph, dh, lh, _k1 = self._host_ptr(H)
        p1, d1, l1, _k2 = self._host_ptr(H1)
        po, do, lo, _k3 = self._host_ptr(out)
        q1, e1, m1, _k4 = self._host_ptr(out1)
        if d1 != dh or l1 != lh or e1 != do or m1 != lo:
            raise ValueError("H1 / D1 must match the dtype and pitch of H / D")
        r = Sp2Result()
        st = lib.sp2_response_host(self._h, C.c_void_p(ph), C.c_void_p(p1), dh, lh, n, int(n_occ), float(tol),
                                   C.c_void_p(po), C.c_void_p(q1), do, lo, C.byref(r), self._stream())
        self._raise(st)
        return out, out1, r.as_dict()

    def congruence(self, Z, X, transpose_first: bool = True, out=None, out_dtype=None):
        """sp2_congruence: C = Z^T X Z (transpose_first) or Z X Z^T for symmetric X; CUDA tensors in, CUDA tensor out."""
        import torch

        n = X.shape[0]
        self._check_dev(Z, n)
        self._check_dev(X, n)
        if Z.dtype != X.dtype or Z.stride(0) != X.stride(0):
            raise ValueError("Z must have the dtype and pitch of X")
        if out is None:
            out = torch.empty((n, n), dtype=out_dtype or X.dtype, device=X.device)
        self._check_dev(out, n)
        st = lib.sp2_congruence(self._h, C.c_void_p(Z.data_ptr()), C.c_void_p(X.data_ptr()), _dtype_code(X), X.stride(0), n,
                                1 if transpose_first else 0, C.c_void_p(out.data_ptr()), _dtype_code(out), out.stride(0),
                                self._stream())
        self._raise(st)
        return out

    # ------------------------------------------------------------------ sequence calls
    def sequence_begin(self, n: int, n_occ: int, tol: float = 0.0, n_steps_hint: int = 64):
        self._raise(lib.sp2_sequence_begin(self._h, int(n), int(n_occ), float(tol), int(n_steps_hint), self._stream()))
        self._seq_n = int(n)

    def sequence_step(self, H_t, D_t):
        n = self._seq_n
        self._check_dev(H_t, n)
        self._check_dev(D_t, n)
        self._raise(lib.sp2_sequence_step(self._h, C.c_void_p(H_t.data_ptr()), _dtype_code(H_t), H_t.stride(0),
                                          C.c_void_p(D_t.data_ptr()), _dtype_code(D_t), D_t.stride(0)))

    def sequence_end(self):
        res = (Sp2Result * 4096)()
        cnt = C.c_int(0)
        st = lib.sp2_sequence_end(self._h, res, C.byref(cnt))
        out = [res[k].as_dict() for k in range(cnt.value)]
        self._raise(st)
        return out

    # ------------------------------------------------------------------ test hooks
    def debug_layout(self):
        """sp2_debug_layout: list of dicts name / offset / reserved / used (bytes) of the workspace regions."""
        n = lib.sp2_debug_layout(self._h, -1, None, None, None, None)
        out = []
        for k in range(n):
            name = C.create_string_buffer(24)
            off, res, used = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
            lib.sp2_debug_layout(self._h, k, name, C.byref(off), C.byref(res), C.byref(used))
            out.append(dict(name=name.value.decode(), offset=off.value, reserved=res.value, used=used.value))
        return out

    def check_canary(self):
        """With a sentinel-filled workspace: every region's used extent fits its reservation, and every byte the
        calls so far were NOT entitled to write (tails of the regions, padding between them, both guard bands)
        still holds the sentinel.  Returns the list of violations (empty = clean)."""
        import torch

        assert self.sentinel is not None, "create the handle with sentinel=<byte>"
        torch.cuda.synchronize(self.device)
        bad = []
        ws = self.workspace
        regions = sorted(self.debug_layout(), key=lambda r: r["offset"])

        def intact(lo, hi, what):     # [lo, hi) relative to the tensor start
            if hi > lo and not bool((ws[lo:hi] == self.sentinel).all()):
                first = int((ws[lo:hi] != self.sentinel).nonzero()[0]) + lo
                bad.append(f"{what}: byte {first - self._ws_off} of the workspace was written")

        intact(0, self._ws_off, "guard band before the workspace")
        cursor = 0
        for r in regions:
            if r["used"] > r["reserved"]:
                bad.append(f"{r['name']}: used {r['used']} > reserved {r['reserved']}")
            intact(self._ws_off + cursor, self._ws_off + r["offset"], f"gap before {r['name']}")
            intact(self._ws_off + r["offset"] + min(r["used"], r["reserved"]), self._ws_off + r["offset"] + r["reserved"],
                   f"tail of {r['name']}")
            cursor = r["offset"] + r["reserved"]
        intact(self._ws_off + cursor, ws.numel(), "after the last region")
        return bad

    def debug_history(self):
        tr = (C.c_double * 128)()
        e = (C.c_double * 128)()
        cnt = lib.sp2_debug_history(self._h, tr, e, 128)
        return list(tr[:cnt]), list(e[:cnt])

    def debug_plane(self, which: int):
        """Internal FP16 plane of the final iterate as a torch view: (tensor[npad, npad], exponent, shift c)."""
        import torch

        off, pitch, ex, sh = C.c_size_t(0), C.c_long(0), C.c_int(0), C.c_double(0)
        self._raise(lib.sp2_debug_plane(self._h, int(which), C.byref(off), C.byref(pitch), C.byref(ex), C.byref(sh)))
        npad = pitch.value
        start = self._ws_off + off.value
        raw = self.workspace[start:start + npad * npad * 2]
        return raw.view(torch.float16).view(npad, npad), ex.value, sh.value
