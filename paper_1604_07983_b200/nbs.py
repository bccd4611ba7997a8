"""Thin Python binding over the C-ABI library (include/nbs.h).  Argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind `libnbs.so`; PyTorch supplies device
memory (`torch.Tensor.data_ptr()`) and streams (`torch.cuda.Stream.cuda_stream`).  There is no CPU
fallback: if the library cannot be built or loaded, or no CUDA device is usable, calls raise.

Function names follow the C ABI (nbs_create / nbs_load_propagators / nbs_correlator /
nbs_destroy, BASELINE.json north_star); `Nbs` is a small convenience class over them.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_longlong, c_size_t, c_void_p

from . import build as _build

NBS_P, NBS_N, NBS_LAMBDA, NBS_SIGMA_P, NBS_SIGMA_0, NBS_SIGMA_M, NBS_XI_0, NBS_XI_M = range(8)
NBS_XU, NBS_XD, NBS_XS = 8, 9, 10
NBS_OK, NBS_EINVAL, NBS_ENOMEM, NBS_ESTATE, NBS_ECUDA = 0, -1, -2, -3, -4
NBS_MEM_DEVICE, NBS_MEM_HOST = 0, 1
STATIC_SCRATCH_BYTES = 32 << 20  # NBS_STATIC_SCRATCH_BYTES (include/nbs.h)

# short names used by the tests and the oracle's channel tuples
BARYON_ID = {"p": NBS_P, "n": NBS_N, "L": NBS_LAMBDA, "Sp": NBS_SIGMA_P, "S0": NBS_SIGMA_0, "Sm": NBS_SIGMA_M,
             "X0": NBS_XI_0, "Xm": NBS_XI_M, "Xu": NBS_XU, "Xd": NBS_XD, "Xs": NBS_XS}
BARYON_NAME = {v: k for k, v in BARYON_ID.items()}

EXPORTS = ["nbs_create", "nbs_load_propagators", "nbs_correlator", "nbs_destroy", "nbs_last_error",
           "nbs_workspace_bytes", "nbs_num_channels", "nbs_channel_info", "nbs_std_channels",
           "nbs_diagram_stats", "nbs_blocks_x", "nbs_model_flops", "nbs_exec_flops", "nbs_fft3d",
           "nbs_kernel_launches", "nbs_set_timing", "nbs_stage_times", "nbs_set_direct", "nbs_set_pipelined", "nbs_num_slots",
           "nbs_probe_fp64", "nbs_probe_kstep", "nbs_tiled_info", "nbs_pair_order", "nbs_plan_selfcheck",
           "nbs_blocks_x_static", "nbs_set_channel_relations", "nbs_iso_relations"]


class nbs_channel(ctypes.Structure):
    _fields_ = [("b1", c_int), ("b2", c_int), ("b3", c_int), ("b4", c_int)]


class NbsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"nbs error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load (building if stale) libnbs.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.ensure_built()
        L = ctypes.CDLL(path)
        L.nbs_create.argtypes = [POINTER(c_void_p), c_int, c_int, POINTER(nbs_channel), c_int, c_int, c_size_t]
        L.nbs_load_propagators.argtypes = [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_int, c_void_p]
        L.nbs_correlator.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_size_t, c_int, c_void_p]
        L.nbs_destroy.argtypes = [c_void_p]
        L.nbs_destroy.restype = None
        L.nbs_last_error.argtypes = [c_void_p]
        L.nbs_last_error.restype = c_char_p
        L.nbs_workspace_bytes.argtypes = [c_void_p]
        L.nbs_workspace_bytes.restype = c_size_t
        L.nbs_num_channels.argtypes = [c_void_p]
        L.nbs_channel_info.argtypes = [c_void_p, c_int, POINTER(nbs_channel)]
        L.nbs_std_channels.argtypes = [POINTER(nbs_channel), c_int]
        L.nbs_diagram_stats.argtypes = [POINTER(nbs_channel), POINTER(c_int), POINTER(c_int), c_int,
                                        POINTER(c_longlong)]
        L.nbs_blocks_x.argtypes = [c_void_p, c_int, c_int, c_void_p, c_size_t, c_void_p]
        L.nbs_blocks_x_static.argtypes = [c_void_p, c_int, c_int, c_void_p, c_size_t, c_void_p]
        L.nbs_model_flops.argtypes = [c_void_p, POINTER(c_double), POINTER(c_double), POINTER(c_double)]
        L.nbs_exec_flops.argtypes = [c_void_p, POINTER(c_double)]
        L.nbs_fft3d.argtypes = [c_void_p, c_void_p, c_size_t, c_int, c_void_p]
        L.nbs_set_timing.argtypes = [c_void_p, c_int]
        L.nbs_set_direct.argtypes = [c_void_p, c_int]
        L.nbs_set_pipelined.argtypes = [c_void_p, c_int]
        L.nbs_set_channel_relations.argtypes = [c_void_p, c_int]
        L.nbs_iso_relations.argtypes = [POINTER(nbs_channel), c_int, POINTER(c_int), POINTER(c_int), POINTER(c_int), c_int]
        L.nbs_stage_times.argtypes = [c_void_p, POINTER(c_double), POINTER(c_longlong), c_int]
        L.nbs_kernel_launches.argtypes = [c_void_p]
        L.nbs_num_slots.argtypes = [c_void_p]
        L.nbs_plan_selfcheck.argtypes = [POINTER(nbs_channel), c_int]
        L.nbs_pair_order.argtypes = [c_void_p, POINTER(c_int), POINTER(c_int), c_int]
        L.nbs_tiled_info.argtypes = [c_void_p, POINTER(c_int), POINTER(c_longlong)]
        L.nbs_probe_fp64.argtypes = [c_void_p, c_int, c_int, POINTER(c_double), POINTER(c_double)]
        L.nbs_probe_kstep.argtypes = [c_void_p, c_int, c_int, c_int, c_int, POINTER(c_double), POINTER(c_double)]
        L.nbs_kernel_launches.restype = c_longlong
        _lib = L
    return _lib


def _check(ctx, rc: int) -> int:
    if rc < 0:
        raise NbsError(rc, lib().nbs_last_error(ctx).decode())
    return rc


def _as_channels(channels):
    arr = (nbs_channel * len(channels))()
    for i, ch in enumerate(channels):
        ids = [BARYON_ID[b] if isinstance(b, str) else int(b) for b in ch]
        arr[i] = nbs_channel(*ids)
    return arr


# --------------------------------------------------------------------------------------------
# host-only helpers (no CUDA call): the table generator's statistics
# --------------------------------------------------------------------------------------------
def nbs_std_channels() -> list[tuple[str, str, str, str]]:
    buf = (nbs_channel * 64)()
    n = lib().nbs_std_channels(buf, 64)
    return [tuple(BARYON_NAME[x] for x in (buf[i].b1, buf[i].b2, buf[i].b3, buf[i].b4)) for i in range(n)]


def nbs_plan_selfcheck(channels=None) -> int:
    """Host-only bounds check of the kernel tables (0 = all invariants hold)."""
    if channels is None:
        return lib().nbs_plan_selfcheck(None, 0)
    arr = _as_channels(channels)
    return lib().nbs_plan_selfcheck(arr, len(channels))


def nbs_iso_relations(channels=None) -> list:
    """Host-only: [(from, sign, swap34)] per channel; from = -1 for a computed channel (include/nbs.h)."""
    n = 52 if channels is None else len(channels)
    arr = None if channels is None else _as_channels(channels)
    fr, sg, sw = (c_int * n)(), (c_int * n)(), (c_int * n)()
    got = lib().nbs_iso_relations(arr, 0 if channels is None else n, fr, sg, sw, n)
    if got < 0:
        raise NbsError(got, "invalid channel list")
    return [(fr[i], sg[i], sw[i]) for i in range(got)]


def nbs_diagram_stats(channel) -> dict:
    ch = _as_channels([channel])
    K = (c_int * 4096)()
    sg = (c_int * 4096)()
    lit = c_longlong(0)
    n = _check(None, lib().nbs_diagram_stats(ch, K, sg, 4096, byref(lit)))
    return dict(diagrams=n, K=list(K[:n]), sign=list(sg[:n]), literal_terms=lit.value)


# --------------------------------------------------------------------------------------------
# the four calls of the boundary
# --------------------------------------------------------------------------------------------
def nbs_create(L: int, T: int, channels=None, device: int = 0, workspace_budget_bytes: int = 0) -> c_void_p:
    ctx = c_void_p()
    if channels is None:
        rc = lib().nbs_create(byref(ctx), L, T, None, 0, device, workspace_budget_bytes)
    else:
        arr = _as_channels(channels)
        rc = lib().nbs_create(byref(ctx), L, T, arr, len(channels), device, workspace_budget_bytes)
    _check(None, rc)
    return ctx


def _ptr_and_loc(x):
    """torch tensor (cuda or cpu) or numpy array -> (pointer, memloc, keepalive)."""
    import numpy as np
    if isinstance(x, np.ndarray):
        assert x.dtype == np.complex128 and x.flags.c_contiguous
        return x.ctypes.data, NBS_MEM_HOST
    import torch
    assert isinstance(x, torch.Tensor) and x.dtype == torch.complex128 and x.is_contiguous()
    return x.data_ptr(), (NBS_MEM_DEVICE if x.is_cuda else NBS_MEM_HOST)


def _stream_handle(stream) -> c_void_p:
    if stream is None:
        import torch
        return c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return c_void_p(stream.cuda_stream)
    return c_void_p(int(stream))


def nbs_load_propagators(ctx, t: int, u, d, s, stream=None) -> None:
    pu, lu = _ptr_and_loc(u)
    pd, ld = _ptr_and_loc(d)
    ps, ls = _ptr_and_loc(s)
    if not (lu == ld == ls):
        raise ValueError("u, d, s must all be device tensors or all be host arrays")
    _check(ctx, lib().nbs_load_propagators(ctx, t, pu, pd, ps, lu, _stream_handle(stream)))


def nbs_correlator(ctx, t: int, ch_begin: int, ch_end: int, out, stream=None) -> None:
    po, lo = _ptr_and_loc(out)
    nbytes = out.nbytes if hasattr(out, "nbytes") else out.numel() * out.element_size()
    _check(ctx, lib().nbs_correlator(ctx, t, ch_begin, ch_end, po, nbytes, lo, _stream_handle(stream)))


def nbs_destroy(ctx) -> None:
    lib().nbs_destroy(ctx)


class Nbs:
    """Context manager over the C ABI.  F = Nbs(L, T).load(t, u, d, s).correlator(t)."""

    def __init__(self, L: int, T: int, channels=None, device: int = 0, workspace_budget_bytes: int = 0):
        self.L, self.T, self.V, self.device = L, T, L ** 3, device
        self.ctx = nbs_create(L, T, channels, device, workspace_budget_bytes)
        self.nch = lib().nbs_num_channels(self.ctx)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def close(self):
        if self.ctx is not None:
            nbs_destroy(self.ctx)
            self.ctx = None

    def channels(self):
        out = []
        for i in range(self.nch):
            ch = nbs_channel()
            _check(self.ctx, lib().nbs_channel_info(self.ctx, i, byref(ch)))
            out.append(tuple(BARYON_NAME[x] for x in (ch.b1, ch.b2, ch.b3, ch.b4)))
        return out

    def load(self, t, u, d, s, stream=None):
        nbs_load_propagators(self.ctx, t, u, d, s, stream)
        return self

    def correlator(self, t, ch_begin=0, ch_end=None, out=None, stream=None):
        import torch
        ch_end = self.nch if ch_end is None else ch_end
        if out is None:
            out = torch.empty((ch_end - ch_begin, 4, 4, 4, 4, self.V), dtype=torch.complex128,
                              device=f"cuda:{self.device}")
        nbs_correlator(self.ctx, t, ch_begin, ch_end, out, stream)
        return out

    def blocks_x(self, t, baryon, stream=None):
        import torch
        b = BARYON_ID[baryon] if isinstance(baryon, str) else int(baryon)
        out = torch.empty((self.V, 4, 12, 12, 12), dtype=torch.complex128, device=f"cuda:{self.device}")
        _check(self.ctx, lib().nbs_blocks_x(self.ctx, t, b, out.data_ptr(), out.numel() * 16, _stream_handle(stream)))
        return out

    def blocks_x_static(self, t, baryon, out, stream=None):
        """nbs_blocks_x_static: eq. 4.1 into the caller's tensor `out` [V][4][12][12][12] complex128, staged rows in
        the library's static scratch array (STATIC_SCRATCH_BYTES); no device memory is allocated."""
        b = BARYON_ID[baryon] if isinstance(baryon, str) else int(baryon)
        assert out.is_cuda and out.is_contiguous()
        _check(self.ctx, lib().nbs_blocks_x_static(self.ctx, t, b, out.data_ptr(), out.numel() * out.element_size(),
                                                   _stream_handle(stream)))
        return out

    def fft3d(self, data, inverse=False, stream=None):
        """In-place 3-D FFT of a device tensor [V][R] complex128 (site-major), rows a2/a5."""
        assert data.is_cuda and data.is_contiguous() and data.shape[0] == self.V
        R = data.numel() // self.V
        _check(self.ctx, lib().nbs_fft3d(self.ctx, data.data_ptr(), R, 1 if inverse else 0, _stream_handle(stream)))
        return data

    def model_flops(self) -> dict:
        b, f, p = c_double(), c_double(), c_double()
        _check(self.ctx, lib().nbs_model_flops(self.ctx, byref(b), byref(f), byref(p)))
        e = c_double()
        _check(self.ctx, lib().nbs_exec_flops(self.ctx, byref(e)))
        return dict(blocks=b.value, fft=f.value, product=p.value, product_executed=e.value)

    STAGES = ("blocks", "fft_fwd", "product", "fft_inv", "output")

    def set_direct(self, enable: bool = True):
        """nbs_set_direct: eq. 2.4 as a shifted sum in x-space (tiny lattices, L <= 8)."""
        _check(self.ctx, lib().nbs_set_direct(self.ctx, 1 if enable else 0))

    def set_pipelined(self, enable: bool = True):
        """nbs_set_pipelined: choose the pipelined product kernel (compact blocks, default) or the one-buffer one."""
        _check(self.ctx, lib().nbs_set_pipelined(self.ctx, 1 if enable else 0))

    def pipelined(self) -> bool:
        return bool(_check(self.ctx, lib().nbs_set_pipelined(self.ctx, -1)))

    def set_channel_relations(self, enable: bool = True):
        """nbs_set_channel_relations: in the isospin limit (d is u) write the u <-> d images of channels from their originals."""
        _check(self.ctx, lib().nbs_set_channel_relations(self.ctx, 1 if enable else 0))

    def derived_channels(self) -> int:
        """Number of channels the isospin limit derives from others (0: none, not available, or switched off)."""
        return int(_check(self.ctx, lib().nbs_set_channel_relations(self.ctx, -1)))

    def conjugate_pairs(self) -> int:
        """Number of sink pairs (a field and its u <-> d image) the isospin limit contracts for half of the momenta."""
        return int(_check(self.ctx, lib().nbs_set_channel_relations(self.ctx, -2)))

    def set_timing(self, enable: bool = True):
        _check(self.ctx, lib().nbs_set_timing(self.ctx, 1 if enable else 0))

    def stage_times(self, reset: bool = True) -> dict:
        """{stage: (total ms, timed executions)} from CUDA events on the launching streams."""
        ms = (c_double * len(self.STAGES))()
        calls = (c_longlong * len(self.STAGES))()
        _check(self.ctx, lib().nbs_stage_times(self.ctx, ms, calls, 1 if reset else 0))
        return {name: (ms[i], calls[i]) for i, name in enumerate(self.STAGES)}

    def tiled_info(self) -> dict:
        """nbs_tiled_info: {tiled, chunk_slots, chunk_builds}."""
        n, b = c_int(), c_longlong()
        t = _check(self.ctx, lib().nbs_tiled_info(self.ctx, byref(n), byref(b)))
        return dict(tiled=bool(t), chunk_slots=n.value, chunk_builds=b.value)

    def pair_order(self) -> list:
        """nbs_pair_order: [(ch_begin, ch_end)] per sink pair, in the library's walking order."""
        lo, hi = (c_int * 64)(), (c_int * 64)()
        n = _check(self.ctx, lib().nbs_pair_order(self.ctx, lo, hi, 64))
        return [(lo[i], hi[i]) for i in range(min(n, 64))]

    def num_slots(self) -> int:
        return _check(self.ctx, lib().nbs_num_slots(self.ctx))

    def probe_kstep(self, cls: int, warps: int, nsteps: int = 18, reps: int = 200) -> dict:
        """nbs_probe_kstep: {cycles, cycles_max, per_subpartition} per k-step of the product kernel's unit code in isolation."""
        avg, mx = c_double(), c_double()
        _check(self.ctx, lib().nbs_probe_kstep(self.ctx, cls, warps, nsteps, reps, byref(avg), byref(mx)))
        return dict(cycles=avg.value, cycles_max=mx.value, per_subpartition=avg.value / (warps / 4.0))

    def probe_fp64(self, mode: int, iters: int = 20000) -> dict:
        """nbs_probe_fp64: {tflops, ms} of a register-resident FP64 instruction mix (see include/nbs.h)."""
        tf, ms = c_double(), c_double()
        _check(self.ctx, lib().nbs_probe_fp64(self.ctx, mode, iters, byref(tf), byref(ms)))
        return dict(tflops=tf.value, ms=ms.value)

    def workspace_bytes(self) -> int:
        return lib().nbs_workspace_bytes(self.ctx)

    def kernel_launches(self) -> int:
        return lib().nbs_kernel_launches(self.ctx)
