"""Thin Python binding of libcwo.so (include/cwo.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and
streams.  There is no CPU fallback: if libcwo.so cannot be loaded this module raises.

    plan = cwo_plan(Nx, Ny, pitch, lam)
    cwo_asm(plan, u1, u2, z)                     # u1, u2: torch.complex64 CUDA tensors [Ny, Nx]
    cwo_fresnel_conv(plan, u1, u2, z)
    cwo_fresnel_fourier(plan, u1, u2, z)         # destination pitch lam |z| / (N pitch)
    cwo_fresnel_shifted(plan, u1, u2, z)         # destination pitch / offset: plan.set_dst_pitch_xy, plan.set_offset
    cwo_propagate_stack(plan, u1, zs, out)       # out: [n, Ny, Nx]
    cwo_gs(plan, amp_src, amp_dst, z, iters, phase)   # phase: float32 in/out
"""
from __future__ import annotations

import ctypes
import os
from typing import Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("CWO_LIBRARY_PATH") or os.path.join(_HERE, "libcwo.so")

CWO_OK, CWO_EINVAL, CWO_EWORKSPACE, CWO_EUNSUPPORTED, CWO_ECUDA, CWO_ENOMEM, CWO_ELIMIT = 0, -1, -2, -3, -4, -5, -6
CWO_SCALE255_STATIC_MAX_N = 1 << 28
CWO_OP_ASM, CWO_OP_FRESNEL, CWO_OP_STACK, CWO_OP_GS, CWO_OP_FRESNEL_FOURIER, CWO_OP_FRESNEL_SHIFTED = 1, 2, 3, 4, 5, 6
CWO_OPT_GS_METHOD = 1
CWO_OPT_PIPELINE = 3
CWO_OPT_ASM_PAD2X = 5
CWO_OPT_STACK_INTENSITY = 6
CWO_OPT_ASM_BAND_LIMIT = 7
CWO_OPT_OUT_REAL = 8
CWO_OUT_COMPLEX, CWO_OUT_INTENSITY, CWO_OUT_AMPLITUDE, CWO_OUT_RE, CWO_OUT_IM, CWO_OUT_PHASE = 0, 1, 2, 3, 4, 5
CWO_GS_FRESNEL, CWO_GS_ASM = 0, 1

# include/cwo.h (the product boundary) and include/cwo_debug.h (measurement hooks of the harness)
EXPORTS = ["cwo_plan", "cwo_plan_destroy", "cwo_plan_set_stream", "cwo_plan_set_pitch_xy", "cwo_plan_set_option",
           "cwo_plan_set_offset", "cwo_plan_set_dst_pitch_xy", "cwo_plan_workspace_bytes", "cwo_plan_set_workspace",
           "cwo_asm", "cwo_fresnel_conv", "cwo_fresnel_fourier", "cwo_fresnel_shifted", "cwo_propagate_stack", "cwo_gs",
           "cwo_scale255", "cwo_scale255_static", "cwo_pls_cgh", "cwo_strerror", "cwo_last_cuda_error"]
DEBUG_EXPORTS = ["cwo_debug_set_timing", "cwo_debug_timings", "cwo_debug_launch_count", "cwo_debug_set_fresnel_2d",
                 "cwo_debug_set_fresnel_gather"]

_lib = None


class CwoError(RuntimeError):
    def __init__(self, code: int, what: str, cuda: int = 0):
        self.code = code
        msg = "%s: %s" % (what, lib().cwo_strerror(code).decode())
        if code == CWO_ECUDA:
            msg += " (cudaError %d)" % cuda
        super().__init__(msg)


def lib() -> ctypes.CDLL:
    """Load libcwo.so (built in-tree by paper_1107_5578_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("libcwo.so is missing (%s): run `python -m paper_1107_5578_b200.build`; "
                          "there is no CPU fallback" % _LIB_PATH)
    L = ctypes.CDLL(_LIB_PATH)
    vp, I, D, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    L.cwo_plan.argtypes = [I, I, D, D, ctypes.POINTER(vp)]
    L.cwo_plan_destroy.argtypes = [vp]
    L.cwo_plan_set_stream.argtypes = [vp, vp]
    L.cwo_plan_set_pitch_xy.argtypes = [vp, D, D]
    L.cwo_plan_set_option.argtypes = [vp, I, I]
    L.cwo_plan_set_offset.argtypes = [vp, D, D]
    L.cwo_plan_set_dst_pitch_xy.argtypes = [vp, D, D]
    L.cwo_plan_workspace_bytes.argtypes = [vp, I, I]
    L.cwo_plan_workspace_bytes.restype = sz
    L.cwo_plan_set_workspace.argtypes = [vp, vp, sz]
    L.cwo_asm.argtypes = [vp, vp, vp, D]
    L.cwo_fresnel_conv.argtypes = [vp, vp, vp, D]
    L.cwo_fresnel_fourier.argtypes = [vp, vp, vp, D]
    L.cwo_fresnel_shifted.argtypes = [vp, vp, vp, D]
    L.cwo_propagate_stack.argtypes = [vp, vp, ctypes.POINTER(D), I, vp]
    L.cwo_gs.argtypes = [vp, vp, vp, D, I, vp]
    L.cwo_scale255.argtypes = [vp, vp, vp, sz]
    L.cwo_scale255_static.argtypes = [vp, vp, sz, vp, ctypes.POINTER(I)]
    L.cwo_pls_cgh.argtypes = [vp, vp, I, vp]
    L.cwo_strerror.argtypes = [I]
    L.cwo_strerror.restype = ctypes.c_char_p
    L.cwo_last_cuda_error.argtypes = [vp]
    L.cwo_debug_launch_count.argtypes = [vp]
    L.cwo_debug_launch_count.restype = ctypes.c_longlong
    L.cwo_debug_timings.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(I), I]
    L.cwo_debug_set_timing.argtypes = [vp, I]
    L.cwo_debug_set_fresnel_2d.argtypes = [vp, I]
    L.cwo_debug_set_fresnel_gather.argtypes = [vp, I]
    _lib = L
    return L


class Plan:
    """Owns a cwo_plan_t and (optionally) a torch-allocated workspace handed to the library."""

    def __init__(self, Nx: int, Ny: int, pitch: float, lam: float):
        self.Nx, self.Ny = int(Nx), int(Ny)
        self._h = ctypes.c_void_p()
        self._ws = None
        self._ws_streams = set()      # streams (handles) the current workspace tensor has been recorded on
        self.stack_intensity = False
        self.out_real = False         # CWO_OPT_OUT_REAL set: u2 of the single-propagation calls is float32
        rc = lib().cwo_plan(self.Nx, self.Ny, float(pitch), float(lam), ctypes.byref(self._h))
        if rc != CWO_OK:
            raise CwoError(rc, "cwo_plan")

    def _check(self, rc: int, what: str) -> None:
        if rc != CWO_OK:
            raise CwoError(rc, what, lib().cwo_last_cuda_error(self._h))

    def set_pitch_xy(self, px: float, py: float) -> None:
        self._check(lib().cwo_plan_set_pitch_xy(self._h, float(px), float(py)), "cwo_plan_set_pitch_xy")

    def set_option(self, key: int, value: int) -> None:
        self._check(lib().cwo_plan_set_option(self._h, int(key), int(value)), "cwo_plan_set_option")
        if key == CWO_OPT_STACK_INTENSITY:
            self.stack_intensity = bool(value)
        if key == CWO_OPT_OUT_REAL:
            self.out_real = bool(value)

    def set_offset(self, ox: float, oy: float) -> None:
        self._check(lib().cwo_plan_set_offset(self._h, float(ox), float(oy)), "cwo_plan_set_offset")

    def set_dst_pitch_xy(self, p1x: float, p1y: float) -> None:
        self._check(lib().cwo_plan_set_dst_pitch_xy(self._h, float(p1x), float(p1y)), "cwo_plan_set_dst_pitch_xy")

    # include/cwo_debug.h: measurement hooks (harness only)
    def set_timing(self, on: bool) -> None:
        self._check(lib().cwo_debug_set_timing(self._h, int(bool(on))), "cwo_debug_set_timing")

    def set_fresnel_2d(self, on: bool) -> None:
        self._check(lib().cwo_debug_set_fresnel_2d(self._h, int(bool(on))), "cwo_debug_set_fresnel_2d")

    def set_fresnel_gather(self, mode: int) -> None:
        self._check(lib().cwo_debug_set_fresnel_gather(self._h, int(mode)), "cwo_debug_set_fresnel_gather")

    def workspace_bytes(self, op: int, n: int = 0) -> int:
        return int(lib().cwo_plan_workspace_bytes(self._h, int(op), int(n)))

    def set_workspace(self, t: "torch.Tensor | None") -> None:
        self._ws = t
        self._ws_streams = set()
        if t is None:
            self._check(lib().cwo_plan_set_workspace(self._h, None, 0), "cwo_plan_set_workspace")
        else:
            self._check(lib().cwo_plan_set_workspace(self._h, t.data_ptr(), t.numel() * t.element_size()),
                        "cwo_plan_set_workspace")

    def ensure_workspace(self, op: int, n: int = 0) -> None:
        need = self.workspace_bytes(op, n)
        have = 0 if self._ws is None else self._ws.numel() * self._ws.element_size()
        if have < need:
            # Kernels already enqueued may still use the old block.  bind_stream() has recorded it on every stream the
            # plan was bound to while it was the workspace, so the caching allocator keeps it back until those streams
            # have passed this point, whichever stream is current now.
            self.set_workspace(torch.empty(need, dtype=torch.uint8, device="cuda"))

    def bind_stream(self) -> None:
        st = torch.cuda.current_stream()
        self._check(lib().cwo_plan_set_stream(self._h, st.cuda_stream), "cwo_plan_set_stream")
        # the call about to be enqueued on `st` uses the workspace, which torch may have allocated under another stream
        if self._ws is not None and st.cuda_stream not in self._ws_streams:
            self._ws.record_stream(st)
            self._ws_streams.add(st.cuda_stream)

    def timings(self, cap: int = 4096):
        """[(tag, ms), ...] of the pass kernels launched since timing was switched on / last read."""
        ms = (ctypes.c_float * cap)(); tag = (ctypes.c_int * cap)()
        n = lib().cwo_debug_timings(self._h, ms, tag, cap)
        if n < 0:
            self._check(n, "cwo_debug_timings")
        return [(int(tag[i]), float(ms[i])) for i in range(min(n, cap))]

    @property
    def launch_count(self) -> int:
        return int(lib().cwo_debug_launch_count(self._h))

    def close(self) -> None:
        if self._h:
            lib().cwo_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _field(t: torch.Tensor, dtype, shape, name: str) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
            and tuple(t.shape) == tuple(shape)):
        raise TypeError("%s must be a contiguous CUDA %s tensor of shape %s" % (name, dtype, tuple(shape)))
    return t.data_ptr()


def cwo_plan(Nx: int, Ny: int, pitch: float, lam: float) -> Plan:
    return Plan(Nx, Ny, pitch, lam)


def cwo_asm(plan: Plan, u1: torch.Tensor, u2: torch.Tensor, z: float) -> None:
    s = (plan.Ny, plan.Nx)
    a, b = _field(u1, torch.complex64, s, "u1"), _field(u2, torch.float32 if plan.out_real else torch.complex64, s, "u2")
    plan.ensure_workspace(CWO_OP_ASM); plan.bind_stream()
    plan._check(lib().cwo_asm(plan._h, a, b, float(z)), "cwo_asm")


def cwo_fresnel_conv(plan: Plan, u1: torch.Tensor, u2: torch.Tensor, z: float) -> None:
    s = (plan.Ny, plan.Nx)
    a, b = _field(u1, torch.complex64, s, "u1"), _field(u2, torch.float32 if plan.out_real else torch.complex64, s, "u2")
    plan.ensure_workspace(CWO_OP_FRESNEL); plan.bind_stream()
    plan._check(lib().cwo_fresnel_conv(plan._h, a, b, float(z)), "cwo_fresnel_conv")


def cwo_fresnel_fourier(plan: Plan, u1: torch.Tensor, u2: torch.Tensor, z: float) -> None:
    s = (plan.Ny, plan.Nx)
    a, b = _field(u1, torch.complex64, s, "u1"), _field(u2, torch.float32 if plan.out_real else torch.complex64, s, "u2")
    plan.ensure_workspace(CWO_OP_FRESNEL_FOURIER); plan.bind_stream()
    plan._check(lib().cwo_fresnel_fourier(plan._h, a, b, float(z)), "cwo_fresnel_fourier")


def cwo_fresnel_shifted(plan: Plan, u1: torch.Tensor, u2: torch.Tensor, z: float) -> None:
    s = (plan.Ny, plan.Nx)
    a, b = _field(u1, torch.complex64, s, "u1"), _field(u2, torch.float32 if plan.out_real else torch.complex64, s, "u2")
    plan.ensure_workspace(CWO_OP_FRESNEL_SHIFTED); plan.bind_stream()
    plan._check(lib().cwo_fresnel_shifted(plan._h, a, b, float(z)), "cwo_fresnel_shifted")


def cwo_propagate_stack(plan: Plan, u1: torch.Tensor, zs: Sequence[float], out: torch.Tensor) -> None:
    n = len(zs)
    a = _field(u1, torch.complex64, (plan.Ny, plan.Nx), "u1")
    b = _field(out, torch.float32 if plan.stack_intensity else torch.complex64, (n, plan.Ny, plan.Nx), "out")
    arr = (ctypes.c_double * n)(*[float(z) for z in zs])
    plan.ensure_workspace(CWO_OP_STACK, n); plan.bind_stream()
    plan._check(lib().cwo_propagate_stack(plan._h, a, arr, n, b), "cwo_propagate_stack")


def cwo_gs(plan: Plan, amp_src: torch.Tensor, amp_dst: torch.Tensor, z: float, iters: int,
           phase: torch.Tensor) -> None:
    s = (plan.Ny, plan.Nx)
    a = _field(amp_src, torch.float32, s, "amp_src")
    b = _field(amp_dst, torch.float32, s, "amp_dst")
    c = _field(phase, torch.float32, s, "phase")
    plan.ensure_workspace(CWO_OP_GS); plan.bind_stream()
    plan._check(lib().cwo_gs(plan._h, a, b, float(z), int(iters), c), "cwo_gs")


def cwo_scale255(plan: Plan, src: torch.Tensor, dst: torch.Tensor) -> None:
    """Scale, Eq.(21): float32 CUDA tensors of equal shape (any shape); dst may be src."""
    if not (src.is_cuda and dst.is_cuda and src.dtype == torch.float32 and dst.dtype == torch.float32
            and src.is_contiguous() and dst.is_contiguous() and src.shape == dst.shape):
        raise TypeError("src, dst must be contiguous CUDA float32 tensors of one shape")
    plan.bind_stream()
    plan._check(lib().cwo_scale255(plan._h, src.data_ptr(), dst.data_ptr(), src.numel()), "cwo_scale255")


def cwo_scale255_static(src: torch.Tensor, dst: torch.Tensor) -> None:
    """Scale, Eq.(21), for callers that must not allocate device memory (no plan: cwo_plan() calls cudaMalloc).

    Same result as cwo_scale255, bit for bit.  The library keeps the per-chunk minima and maxima in a fixed array inside
    libcwo.so, so at most CWO_SCALE255_STATIC_MAX_N (2**28) floats per call; larger tensors raise CwoError(CWO_ELIMIT).
    This binding allocates nothing either: it passes the two data pointers and torch's current stream.  All calls on a
    GPU share that array: keep them ordered on one stream (calls that overlap on the GPU race).  Make the first call on a
    device outside stream capture (it resolves the array's device address once)."""
    if not (src.is_cuda and dst.is_cuda and src.dtype == torch.float32 and dst.dtype == torch.float32
            and src.is_contiguous() and dst.is_contiguous() and src.shape == dst.shape and src.device == dst.device):
        raise TypeError("src, dst must be contiguous CUDA float32 tensors of one shape on one device")
    err = ctypes.c_int(0)
    with torch.cuda.device(src.device):
        rc = lib().cwo_scale255_static(src.data_ptr(), dst.data_ptr(), src.numel(),
                                       torch.cuda.current_stream().cuda_stream, ctypes.byref(err))
    if rc != CWO_OK:
        raise CwoError(rc, "cwo_scale255_static", err.value)


def cwo_pls_cgh(plan: Plan, pts: torch.Tensor, out: torch.Tensor) -> None:
    """CGH of point light sources, Eq.(23): pts float64 CUDA [n, 4] = (x, y, z, A); out float32 [Ny, Nx]."""
    if not (pts.is_cuda and pts.dtype == torch.float64 and pts.is_contiguous() and pts.dim() == 2 and pts.shape[1] == 4):
        raise TypeError("pts must be a contiguous CUDA float64 tensor of shape [n, 4]")
    b = _field(out, torch.float32, (plan.Ny, plan.Nx), "out")
    plan.bind_stream()
    plan._check(lib().cwo_pls_cgh(plan._h, pts.data_ptr(), int(pts.shape[0]), b), "cwo_pls_cgh")


class HostPipeline:
    """Propagate HOST (pinned) fields: step i's host->device copy, its kernels and its device->host copy run
    on three streams over `depth` rotating device buffers, so the copies of neighbouring steps overlap the
    kernels (and each other: the two directions use different copy engines).  Argument marshalling and
    stream plumbing only -- every propagation is one cwo_asm / cwo_fresnel_conv call."""

    def __init__(self, plan: Plan, op: str = "asm", depth: int = 3):
        if op not in ("asm", "fresnel"):
            raise ValueError("op must be 'asm' or 'fresnel'")
        self.plan, self.depth, self.i = plan, int(depth), 0
        self.call = cwo_asm if op == "asm" else cwo_fresnel_conv
        shape = (plan.Ny, plan.Nx)
        self.d_in = [torch.empty(shape, dtype=torch.complex64, device="cuda") for _ in range(self.depth)]
        self.d_out = [torch.empty(shape, dtype=torch.complex64, device="cuda") for _ in range(self.depth)]
        self.s_in, self.s_run, self.s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
        for t in self.d_in + self.d_out:          # allocated under the current stream, used on the private ones
            for st in (self.s_in, self.s_run, self.s_out):
                t.record_stream(st)
        self.ev_in = [torch.cuda.Event() for _ in range(self.depth)]     # H2D of slot k done
        self.ev_run = [torch.cuda.Event() for _ in range(self.depth)]    # kernels of slot k done
        self.ev_out = [torch.cuda.Event() for _ in range(self.depth)]    # D2H of slot k done
        self.used = [False] * self.depth
        plan.ensure_workspace(CWO_OP_ASM if op == "asm" else CWO_OP_FRESNEL)
        if plan._ws is not None:
            plan._ws.record_stream(self.s_run)

    def start_after(self, stream: "torch.cuda.Stream") -> None:
        """Order everything submitted from now on after the work already queued on `stream`."""
        for s in (self.s_in, self.s_run, self.s_out):
            s.wait_stream(stream)

    def submit(self, host_in: torch.Tensor, host_out: torch.Tensor, z: float) -> None:
        k = self.i % self.depth
        self.i += 1
        with torch.cuda.stream(self.s_in):
            if self.used[k]:
                self.s_in.wait_event(self.ev_run[k])          # the kernels that last read d_in[k]
            self.d_in[k].copy_(host_in, non_blocking=True)
            self.ev_in[k].record(self.s_in)
        with torch.cuda.stream(self.s_run):
            self.s_run.wait_event(self.ev_in[k])
            if self.used[k]:
                self.s_run.wait_event(self.ev_out[k])         # the copy that last read d_out[k]
            self.call(self.plan, self.d_in[k], self.d_out[k], z)
            self.ev_run[k].record(self.s_run)
        with torch.cuda.stream(self.s_out):
            self.s_out.wait_event(self.ev_run[k])
            host_out.copy_(self.d_out[k], non_blocking=True)
            self.ev_out[k].record(self.s_out)
        self.used[k] = True

    def join(self, stream: "torch.cuda.Stream") -> None:
        """Make `stream` wait for everything submitted so far (no host synchronisation)."""
        for s in (self.s_in, self.s_run, self.s_out):
            stream.wait_stream(s)
