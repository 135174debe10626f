"""ctypes binding for libxc.so -- same names as include/xc.h, argument marshalling only.

Tensors are torch CUDA tensors (device memory) or pinned CPU tensors (host memory); only their
data pointers and the stream handle cross the boundary.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libxc.so")
LIB_PROFILE_PATH = os.path.join(HERE, "libxc_profile.so")

MAX_T = 65535
NOALLOC_SCRATCH_BYTES = 16 * 1024 * 1024   # XC_NOALLOC_SCRATCH_BYTES: the fixed device array xc_correlate_i4_noalloc unpacks into
NOALLOC_MAX_N = 576                        # XC_NOALLOC_MAX_N
TIMING_WORDS = 6          # uint64 words of the xc_set_timing_buffer buffer
TRACE_WORDS = 3 * 256 * 4  # int64 words of the profiling build's trace buffer
I8_KERNEL_AUTO, I8_KERNEL_TC, I8_KERNEL_SIMT = 0, 1, 2
OPT_I8_KERNEL, OPT_MAX_CTAS, OPT_FORCE_STAGE, OPT_DEBUG_SKIP, OPT_TILE, OPT_PDL, OPT_TSPLIT = 0, 1, 2, 3, 4, 7, 8
OPT_ORIGIN_SHIFT, OPT_F32_KERNEL = 9, 10
F32_KERNEL_AUTO, F32_KERNEL_CUDA_CORES, F32_KERNEL_TC = 0, 1, 2
TILE_AUTO, TILE_1CTA_128x128, TILE_2CTA_256x256 = 0, 1, 3

# every symbol include/xc.h declares
EXPORTED_SYMBOLS = (
    "xc_plan", "xc_destroy", "xc_in_bytes", "xc_in_bytes_f32", "xc_vis_bytes", "xc_n_baselines",
    "xc_workspace_bytes", "xc_set_workspace", "xc_set_option", "xc_correlate", "xc_correlate_acc",
    "xc_correlate_f32", "xc_correlate_pipelined", "xc_correlate_host", "xc_correlate_channels", "xc_integrate",
    "xc_correlate_i4", "xc_correlate_i4_noalloc", "xc_in_bytes_i4", "xc_correlate_host_i4", "xc_tile_count", "xc_tile_get", "xc_t_split", "xc_origin_shift", "xc_origin_shift_plan", "xc_f32_kernel_used", "xc_correlate_f32_channels",
    "xc_set_in_pitch", "xc_in_pitch", "xc_set_in_pitch_f32", "xc_in_pitch_f32", "xc_scratch_pitch", "xc_scratch_in_bytes", "xc_set_timing_buffer",
    "xc_volt_bytes", "xc_cube_bytes", "xc_fengine", "xc_fengine_f32", "xc_fx", "xc_fengine_channels", "xc_fx_channels",
    "xc_tri_index", "xc_tri_inverse", "xc_last_launches", "xc_status_string", "xc_last_cuda_error", "xc_version",
)
# additionally exported by the profiling build only (libxc_profile.so, -DXC_PROFILE)
PROFILE_SYMBOLS = ("xc_debug_set_trace",)


class XcError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        name = lib().xc_status_string(code).decode() if _lib is not None else str(code)
        super().__init__(f"{where}: {name} ({code}){': ' + detail if detail else ''}")
        self.code = code


_lib = None


def load_library(path: str | None = None) -> ctypes.CDLL:
    """Loads libxc.so; raises (never falls back) if it is missing -- build it with
    `python -m paper_1107_4264_b200.build`."""
    global _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built: run `python -m paper_1107_4264_b200.build` "
                                "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    i, p, sz, i64 = ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int64
    pp = ctypes.POINTER(ctypes.c_void_p)
    sig = {
        "xc_plan": (i, [pp, i, i, i, i, i]),
        "xc_destroy": (None, [p]),
        "xc_in_bytes": (sz, [p]), "xc_in_bytes_f32": (sz, [p]), "xc_vis_bytes": (sz, [p]),
        "xc_n_baselines": (sz, [p]), "xc_workspace_bytes": (sz, [p]),
        "xc_set_workspace": (i, [p, p, sz]),
        "xc_set_option": (i, [p, i, i]),
        "xc_correlate": (i, [p, p, p, p]), "xc_correlate_acc": (i, [p, p, p, p]),
        "xc_correlate_f32": (i, [p, p, p, i, p]),
        "xc_correlate_f32_channels": (i, [p, p, p, i, i, i, p]),
        "xc_correlate_i4": (i, [p, p, p, i, p]),
        "xc_correlate_i4_noalloc": (i, [i, i, i, p, p, i, p]),
        "xc_in_bytes_i4": (sz, [p]),
        "xc_correlate_channels": (i, [p, p, p, i, i, i, p]),
        "xc_integrate": (i, [p, p, i, p, p, p, p, p, p]),
        "xc_correlate_pipelined": (i, [p, p, i, p, p, p, p]),
        "xc_correlate_host": (i, [p, p, p, p, p, p]),
        "xc_correlate_host_i4": (i, [p, p, p, p, p, p]),
        "xc_set_in_pitch": (i, [p, sz]), "xc_in_pitch": (sz, [p]),
        "xc_set_in_pitch_f32": (i, [p, sz]), "xc_in_pitch_f32": (sz, [p]),
        "xc_scratch_pitch": (sz, [p]), "xc_scratch_in_bytes": (sz, [p]),
        "xc_set_timing_buffer": (i, [p, p]),
        "xc_t_split": (i, [p]),
        "xc_volt_bytes": (sz, [p]), "xc_cube_bytes": (sz, [p]),
        "xc_fengine": (i, [p, p, ctypes.c_float, p, sz, p]),
        "xc_fengine_f32": (i, [p, p, p, p]),
        "xc_fx": (i, [p, p, ctypes.c_float, p, p, i, p]),
        "xc_fengine_channels": (i, [p, p, ctypes.c_float, p, sz, i, i, p]),
        "xc_fx_channels": (i, [p, p, ctypes.c_float, p, p, i, i, i, p]),
        "xc_tile_count": (i, [p]),
        "xc_f32_kernel_used": (i, [p]),
        "xc_origin_shift": (i, [p, ctypes.POINTER(i), ctypes.POINTER(i)]),
        "xc_origin_shift_plan": (i, [p, ctypes.c_uint64, sz, ctypes.POINTER(i), ctypes.POINTER(i)]),
        "xc_tile_get": (i, [p, i, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i)]),
        "xc_tri_index": (i64, [i64, i64]),
        "xc_tri_inverse": (None, [i64, ctypes.POINTER(i64), ctypes.POINTER(i64)]),
        "xc_last_launches": (i, [p]),
        "xc_status_string": (ctypes.c_char_p, [i]),
        "xc_last_cuda_error": (ctypes.c_char_p, [p]),
        "xc_version": (ctypes.c_char_p, []),
    }
    if hasattr(L, "xc_debug_set_trace"):      # profiling build
        sig["xc_debug_set_trace"] = (i, [p, p])
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype = res
        fn.argtypes = args
    _lib = L
    return L


def lib() -> ctypes.CDLL:
    return _lib if _lib is not None else load_library()


def version() -> str:
    return lib().xc_version().decode()


def tri_index(bx: int, by: int) -> int:
    """g = by(by+1)/2 + bx."""
    return int(lib().xc_tri_index(bx, by))


def tri_inverse(g: int) -> tuple[int, int]:
    """(bx, by) from g (with the integer fix-up)."""
    bx, by = ctypes.c_int64(), ctypes.c_int64()
    lib().xc_tri_inverse(g, ctypes.byref(bx), ctypes.byref(by))
    return int(bx.value), int(by.value)


def shard_channels(F: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous channel range [f_lo, f_hi) of `rank`: channels are independent and
    the paper's multi-GPU plan is to give each GPU different channels, so sharding
    needs no collective.  Sizes differ by at most one."""
    base, rem = divmod(F, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def _stream_handle(stream) -> ctypes.c_void_p:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def correlate_i4_noalloc(x4, vis=None, accumulate=False, stream=None):
    """xc_correlate_i4_noalloc: the 4-bit X-engine for callers that must not allocate device memory (a real-time capture
    loop, a plug-in of an application that owns all device memory, a process whose HBM a caching allocator has already
    claimed).  No plan, no workspace: the library unpacks into a fixed 16 MiB array of its own device image, shared by
    all calls on the device -- calls that overlap on the GPU race.  x4: uint8 CUDA [T][F][N][2] (low nibble re, high
    nibble im); vis: int32 CUDA [F][N(N+1)/2][2][2][2], written or (accumulate) added to.  Passing vis=None lets torch
    allocate the cube, which of course defeats the purpose: hand one in.  Raises XcError(XC_ERR_NO_WORKSPACE) when
    (4N rounded up to 128) * F * T exceeds NOALLOC_SCRATCH_BYTES, XcError(XC_ERR_UNSUPPORTED) for N > NOALLOC_MAX_N."""
    import torch
    if not (isinstance(x4, torch.Tensor) and x4.is_cuda and x4.dtype == torch.uint8 and x4.is_contiguous()
            and x4.dim() == 4 and x4.shape[3] == 2):
        raise ValueError("input must be a contiguous CUDA uint8 tensor of shape [T][F][N][2]")
    T, F, N = (int(d) for d in x4.shape[:3])
    shape = (F, N * (N + 1) // 2, 2, 2, 2)
    if vis is None:
        vis = torch.empty(shape, dtype=torch.int32, device=x4.device)
    if not (isinstance(vis, torch.Tensor) and vis.is_cuda and vis.dtype == torch.int32 and vis.is_contiguous()
            and tuple(vis.shape) == shape):
        raise ValueError(f"vis must be a contiguous CUDA int32 tensor of shape {shape}")
    rc = lib().xc_correlate_i4_noalloc(N, F, T, ctypes.c_void_p(x4.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                       1 if accumulate else 0, _stream_handle(stream))
    if rc != 0:
        pitch = (4 * N + 127) // 128 * 128
        raise XcError(rc, f"xc_correlate_i4_noalloc(N={N}, F={F}, T={T})",
                      f"unpacked block {pitch * F * T} bytes, fixed scratch {NOALLOC_SCRATCH_BYTES} bytes, N limit {NOALLOC_MAX_N}")
    return vis


class Plan:
    """xc_plan(N, P=2, F, T, layout) + the calls of include/xc.h as methods."""

    def __init__(self, N: int, F: int, T: int, P: int = 2, layout: int = 0):
        self._h = ctypes.c_void_p()
        rc = lib().xc_plan(ctypes.byref(self._h), N, P, F, T, layout)
        if rc != 0:
            self._h = ctypes.c_void_p()
            raise XcError(rc, f"xc_plan(N={N}, P={P}, F={F}, T={T})")
        self.N, self.P, self.F, self.T = N, P, F, T
        self.NB = int(lib().xc_n_baselines(self._h))
        self._ws = None

    def close(self) -> None:
        if getattr(self, "_h", None) and self._h.value:
            lib().xc_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    def _check(self, rc: int, where: str) -> None:
        if rc != 0:
            raise XcError(rc, where, lib().xc_last_cuda_error(self._h).decode())

    # sizes ---------------------------------------------------------------------------------
    @property
    def in_bytes(self) -> int:
        return int(lib().xc_in_bytes(self._h))

    @property
    def in_bytes_f32(self) -> int:
        return int(lib().xc_in_bytes_f32(self._h))

    @property
    def vis_bytes(self) -> int:
        return int(lib().xc_vis_bytes(self._h))

    @property
    def workspace_bytes(self) -> int:
        return int(lib().xc_workspace_bytes(self._h))

    @property
    def last_launches(self) -> int:
        return int(lib().xc_last_launches(self._h))

    def in_shape(self):
        return (self.T, self.F, self.N, 2, 2)

    def vis_shape(self):
        return (self.F, self.NB, 2, 2, 2)

    # options / schedule --------------------------------------------------------------------
    def set_option(self, option: int, value: int) -> None:
        self._check(lib().xc_set_option(self._h, option, value), "xc_set_option")

    def set_workspace(self, ws) -> None:
        """ws: torch uint8/int8 CUDA tensor of at least workspace_bytes (kept alive by the plan)."""
        self._check(lib().xc_set_workspace(self._h, ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()),
                    "xc_set_workspace")
        self._ws = ws

    def tiles(self):
        """[(bi, bj, si, sj)] of the integer path's per-channel tile schedule."""
        out = []
        bi, bj, si, sj = (ctypes.c_int() for _ in range(4))
        for k in range(int(lib().xc_tile_count(self._h))):
            self._check(lib().xc_tile_get(self._h, k, ctypes.byref(bi), ctypes.byref(bj), ctypes.byref(si),
                                          ctypes.byref(sj)), "xc_tile_get")
            out.append((bi.value, bj.value, si.value, sj.value))
        return out

    def set_trace(self, buf) -> None:
        """PROFILING BUILD ONLY (load_library(LIB_PROFILE_PATH)): buf = int64 CUDA tensor of TRACE_WORDS elements or None."""
        if not hasattr(lib(), "xc_debug_set_trace"):
            raise RuntimeError("xc_debug_set_trace exists only in libxc_profile.so (build with --profile)")
        self._check(lib().xc_debug_set_trace(self._h, ctypes.c_void_p(buf.data_ptr() if buf is not None else 0)),
                    "xc_debug_set_trace")
        self._trace = buf

    def set_timing_buffer(self, buf) -> None:
        """buf = CUDA tensor of TIMING_WORDS 64-bit words (or None): see xc_set_timing_buffer.  Preset buf[0] = max, buf[1] = 0
        before each launch; afterwards buf[1] - buf[0] is the kernel's duration in ns."""
        self._check(lib().xc_set_timing_buffer(self._h, ctypes.c_void_p(buf.data_ptr() if buf is not None else 0)),
                    "xc_set_timing_buffer")
        self._stamps = buf

    def set_in_pitch(self, row_pitch_bytes: int) -> None:
        self._check(lib().xc_set_in_pitch(self._h, row_pitch_bytes), "xc_set_in_pitch")

    @property
    def in_pitch(self) -> int:
        return int(lib().xc_in_pitch(self._h))

    def set_in_pitch_f32(self, row_pitch_bytes: int) -> None:
        """Float blocks with rows row_pitch_bytes apart (multiple of 16, >= 16N; 0 = dense): pass them as [T][F][pitch / 4]."""
        self._check(lib().xc_set_in_pitch_f32(self._h, row_pitch_bytes), "xc_set_in_pitch_f32")

    @property
    def in_pitch_f32(self) -> int:
        return int(lib().xc_in_pitch_f32(self._h))

    @property
    def scratch_pitch(self) -> int:
        return int(lib().xc_scratch_pitch(self._h))

    @property
    def scratch_in_bytes(self) -> int:
        return int(lib().xc_scratch_in_bytes(self._h))

    @property
    def t_split(self) -> int:
        return int(lib().xc_t_split(self._h))

    @property
    def f32_kernel_used(self) -> int:
        return int(lib().xc_f32_kernel_used(self._h))

    @property
    def origin_shift(self):
        """[(shift_bytes, tiles)] per channel class f mod P of the last integer compute call (xc_origin_shift)."""
        sh, tl = (ctypes.c_int * 8)(), (ctypes.c_int * 8)()
        n = int(lib().xc_origin_shift(self._h, sh, tl))
        return [(int(sh[c]), int(tl[c])) for c in range(n)]

    def origin_shift_plan(self, base_addr: int, row_pitch_bytes: int):
        """[(shift_bytes, tiles)] per channel class for a block at that address and row pitch (host logic only)."""
        sh, tl = (ctypes.c_int * 8)(), (ctypes.c_int * 8)()
        n = int(lib().xc_origin_shift_plan(self._h, base_addr, row_pitch_bytes, sh, tl))
        return [(int(sh[c]), int(tl[c])) for c in range(n)]

    def new_scratch(self, n: int = 1, device="cuda"):
        """Device scratch for the host-buffer calls: n * scratch_in_bytes int8 (rows re-pitched to 128-byte multiples)."""
        import torch
        return torch.empty(n * self.scratch_in_bytes, dtype=torch.int8, device=device)

    # compute -------------------------------------------------------------------------------
    def _chk_in(self, x, dtype):
        import torch
        ok = isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == dtype and x.is_contiguous()
        if ok and dtype == torch.int8 and tuple(x.shape) == (self.T, self.F, self.in_pitch):
            return                                     # block given as [T][F][row pitch in bytes] (xc_set_in_pitch)
        if ok and dtype == torch.float32 and tuple(x.shape) == (self.T, self.F, self.in_pitch_f32 // 4):
            return                                     # float block given as [T][F][row pitch in floats] (xc_set_in_pitch_f32)
        if ok and dtype == torch.float32 and self.in_pitch_f32 != 16 * self.N:
            raise ValueError(f"pitched float input must be a contiguous CUDA tensor of shape {(self.T, self.F, self.in_pitch_f32 // 4)}")
        if ok and dtype == torch.int8 and self.in_pitch != 4 * self.N:
            raise ValueError(f"pitched input must be a contiguous CUDA int8 tensor of shape {(self.T, self.F, self.in_pitch)}")
        if not (ok and tuple(x.shape) == self.in_shape()):
            raise ValueError(f"input must be a contiguous CUDA {dtype} tensor of shape {self.in_shape()}")

    def _chk_vis(self, v, dtype):
        import torch
        if not (isinstance(v, torch.Tensor) and v.is_cuda and v.dtype == dtype and v.is_contiguous()
                and tuple(v.shape) == self.vis_shape()):
            raise ValueError(f"vis must be a contiguous CUDA {dtype} tensor of shape {self.vis_shape()}")

    def new_vis(self, dtype=None, device="cuda"):
        import torch
        return torch.empty(self.vis_shape(), dtype=dtype or torch.int32, device=device)

    def correlate(self, x, vis=None, stream=None):
        """vis = X-engine(x).  x: int8 CUDA [T][F][N][2][2] -> int32 CUDA [F][NB][2][2][2]."""
        import torch
        self._chk_in(x, torch.int8)
        if vis is None:
            vis = self.new_vis(torch.int32, x.device)
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_correlate(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                       _stream_handle(stream)), "xc_correlate")
        return vis

    def correlate_acc(self, x, vis, stream=None):
        """vis += X-engine(x)."""
        import torch
        self._chk_in(x, torch.int8)
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_correlate_acc(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                           _stream_handle(stream)), "xc_correlate_acc")
        return vis

    def correlate_channels(self, x, vis, f0: int, nf: int, accumulate=False, stream=None):
        """vis[f0:f0+nf] (+)= X-engine(x[:, f0:f0+nf]); x and vis are the plan's full block and cube."""
        import torch
        self._chk_in(x, torch.int8)
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_correlate_channels(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                                f0, nf, 1 if accumulate else 0, _stream_handle(stream)),
                    "xc_correlate_channels")
        return vis

    def correlate_i4(self, x4, vis=None, accumulate=False, stream=None):
        """vis (+)= X-engine(x4) for 4-bit samples.  x4: uint8 CUDA [T][F][N][2] (low nibble re, high nibble im)."""
        import torch
        if not (isinstance(x4, torch.Tensor) and x4.is_cuda and x4.dtype == torch.uint8 and x4.is_contiguous()
                and tuple(x4.shape) == (self.T, self.F, self.N, 2)):
            raise ValueError(f"input must be a contiguous CUDA uint8 tensor of shape {(self.T, self.F, self.N, 2)}")
        if vis is None:
            vis = self.new_vis(torch.int32, x4.device)
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_correlate_i4(self._h, ctypes.c_void_p(x4.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                          1 if accumulate else 0, _stream_handle(stream)), "xc_correlate_i4")
        return vis

    def correlate_f32(self, x, vis=None, accumulate=False, stream=None):
        import torch
        self._chk_in(x, torch.float32)
        if vis is None:
            vis = self.new_vis(torch.float32, x.device)
        self._chk_vis(vis, torch.float32)
        self._check(lib().xc_correlate_f32(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                           1 if accumulate else 0, _stream_handle(stream)), "xc_correlate_f32")
        return vis

    def correlate_f32_channels(self, x, vis, f0: int, nf: int, accumulate=False, stream=None):
        """vis[f0:f0+nf] (+)= X-engine(x[:, f0:f0+nf]) for float samples; x and vis are the plan's full block and cube."""
        import torch
        self._chk_in(x, torch.float32)
        self._chk_vis(vis, torch.float32)
        self._check(lib().xc_correlate_f32_channels(self._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                                    f0, nf, 1 if accumulate else 0, _stream_handle(stream)),
                    "xc_correlate_f32_channels")
        return vis

    def correlate_pipelined(self, blocks_host, dev_buf2, vis, compute_stream, copy_stream):
        """blocks_host: pinned CPU int8 tensor [n_blocks][T][F][N][2][2]; dev_buf2: CUDA int8 tensor of
        2 * scratch_in_bytes; vis: CUDA int32.  Enqueues Algorithm 1 and returns; sync compute_stream."""
        import torch
        if not (blocks_host.dtype == torch.int8 and blocks_host.is_contiguous() and not blocks_host.is_cuda
                and tuple(blocks_host.shape[1:]) == self.in_shape()):
            raise ValueError("blocks_host must be a contiguous CPU int8 tensor [n_blocks][T][F][N][2][2]")
        if dev_buf2.numel() * dev_buf2.element_size() < 2 * self.scratch_in_bytes:
            raise ValueError("dev_buf2 too small")
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_correlate_pipelined(
            self._h, ctypes.c_void_p(blocks_host.data_ptr()), int(blocks_host.shape[0]),
            ctypes.c_void_p(dev_buf2.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
            ctypes.c_void_p(compute_stream.cuda_stream), ctypes.c_void_p(copy_stream.cuda_stream)),
            "xc_correlate_pipelined")
        return vis

    def integrate(self, blocks_host, dev_buf2, vis32, vis64, compute_stream, copy_stream, vis64_host=None):
        """Long integration over pinned host blocks [n_blocks][T][F][N][2][2] into the int64 CUDA cube vis64 (and the
        pinned int64 host cube vis64_host if given).  Enqueues and returns; sync compute_stream."""
        import torch
        if not (blocks_host.dtype == torch.int8 and blocks_host.is_contiguous() and not blocks_host.is_cuda
                and tuple(blocks_host.shape[1:]) == self.in_shape()):
            raise ValueError("blocks_host must be a contiguous CPU int8 tensor [n_blocks][T][F][N][2][2]")
        if dev_buf2.numel() * dev_buf2.element_size() < 2 * self.scratch_in_bytes:
            raise ValueError("dev_buf2 too small")
        self._chk_vis(vis32, torch.int32)
        self._chk_vis(vis64, torch.int64)
        if vis64_host is not None and not (vis64_host.dtype == torch.int64 and vis64_host.is_contiguous()
                                           and tuple(vis64_host.shape) == self.vis_shape() and not vis64_host.is_cuda):
            raise ValueError("vis64_host must be a contiguous CPU int64 tensor of the cube's shape")
        self._check(lib().xc_integrate(
            self._h, ctypes.c_void_p(blocks_host.data_ptr()), int(blocks_host.shape[0]),
            ctypes.c_void_p(dev_buf2.data_ptr()), ctypes.c_void_p(vis32.data_ptr()), ctypes.c_void_p(vis64.data_ptr()),
            ctypes.c_void_p(vis64_host.data_ptr() if vis64_host is not None else 0),
            ctypes.c_void_p(compute_stream.cuda_stream), ctypes.c_void_p(copy_stream.cuda_stream)), "xc_integrate")
        return vis64

    # F-engine + FX chain ---------------------------------------------------------------------
    def volt_shape(self):
        return (self.N, 2, self.T * self.F, 2)

    def _chk_volt(self, volt):
        import torch
        if not (isinstance(volt, torch.Tensor) and volt.is_cuda and volt.dtype == torch.int8 and volt.is_contiguous()
                and tuple(volt.shape) == self.volt_shape()):
            raise ValueError(f"volt must be a contiguous CUDA int8 tensor of shape {self.volt_shape()}")

    def new_cube(self, device="cuda"):
        """int8 [T][F][scratch_pitch]: the F-engine's output / the X-engine's pitched input."""
        import torch
        return torch.empty((self.T, self.F, self.scratch_pitch), dtype=torch.int8, device=device)

    def fengine(self, volt, scale: float, cube=None, stream=None):
        """cube = quantise(FFT_F(volt) * scale) in the X-engine's order.  cube: int8 CUDA [T][F][pitch] (pitch % 4 == 0,
        >= 4N; default new_cube()).  Returns the cube."""
        self._chk_volt(volt)
        if cube is None:
            cube = self.new_cube(volt.device)
        if not (cube.is_cuda and cube.is_contiguous() and cube.dim() == 3 and tuple(cube.shape[:2]) == (self.T, self.F)
                and cube.element_size() == 1):
            raise ValueError("cube must be a contiguous CUDA int8 tensor [T][F][pitch]")
        self._check(lib().xc_fengine(self._h, ctypes.c_void_p(volt.data_ptr()), ctypes.c_float(scale),
                                     ctypes.c_void_p(cube.data_ptr()), int(cube.shape[2]), _stream_handle(stream)), "xc_fengine")
        return cube

    def fengine_f32(self, volt, spec=None, stream=None):
        """Unquantised fp32 spectra, float CUDA [T][F][N][2][2]."""
        import torch
        self._chk_volt(volt)
        if spec is None:
            spec = torch.empty(self.in_shape(), dtype=torch.float32, device=volt.device)
        self._chk_in(spec, torch.float32)
        self._check(lib().xc_fengine_f32(self._h, ctypes.c_void_p(volt.data_ptr()), ctypes.c_void_p(spec.data_ptr()),
                                         _stream_handle(stream)), "xc_fengine_f32")
        return spec

    def fx(self, volt, scale: float, cube_scratch, vis=None, accumulate=False, stream=None):
        """vis (+)= X-engine(F-engine(volt)).  cube_scratch: new_cube()."""
        import torch
        self._chk_volt(volt)
        if tuple(cube_scratch.shape) != (self.T, self.F, self.scratch_pitch) or not cube_scratch.is_contiguous():
            raise ValueError("cube_scratch must be new_cube()")
        if vis is None:
            vis = self.new_vis(torch.int32, volt.device)
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_fx(self._h, ctypes.c_void_p(volt.data_ptr()), ctypes.c_float(scale),
                                ctypes.c_void_p(cube_scratch.data_ptr()), ctypes.c_void_p(vis.data_ptr()),
                                1 if accumulate else 0, _stream_handle(stream)), "xc_fx")
        return vis

    def new_cube_range(self, nf: int, device="cuda"):
        """int8 [T][nf][scratch_pitch]: the pruned cube of a channel range (fengine_channels / fx_channels)."""
        import torch
        return torch.empty((self.T, nf, self.scratch_pitch), dtype=torch.int8, device=device)

    def fengine_channels(self, volt, scale: float, f0: int, nf: int, cube=None, stream=None):
        """Pruned cube [T][nf][pitch] holding channels [f0, f0 + nf) of quantise(FFT_F(volt) * scale)."""
        self._chk_volt(volt)
        if cube is None:
            cube = self.new_cube_range(nf, volt.device)
        if not (cube.is_cuda and cube.is_contiguous() and cube.dim() == 3 and tuple(cube.shape[:2]) == (self.T, nf)
                and cube.element_size() == 1):
            raise ValueError("cube must be a contiguous CUDA int8 tensor [T][nf][pitch]")
        self._check(lib().xc_fengine_channels(self._h, ctypes.c_void_p(volt.data_ptr()), ctypes.c_float(scale),
                                              ctypes.c_void_p(cube.data_ptr()), int(cube.shape[2]), f0, nf, _stream_handle(stream)),
                    "xc_fengine_channels")
        return cube

    def fx_channels(self, volt, scale: float, cube_scratch, vis, f0: int, nf: int, accumulate=False, stream=None):
        """vis[f0:f0+nf] (+)= X-engine(F-engine(volt)[channels f0 .. f0+nf)).  cube_scratch: new_cube_range(nf); vis: the full cube."""
        import torch
        self._chk_volt(volt)
        if tuple(cube_scratch.shape) != (self.T, nf, self.scratch_pitch) or not cube_scratch.is_contiguous():
            raise ValueError("cube_scratch must be new_cube_range(nf)")
        self._chk_vis(vis, torch.int32)
        self._check(lib().xc_fx_channels(self._h, ctypes.c_void_p(volt.data_ptr()), ctypes.c_float(scale),
                                         ctypes.c_void_p(cube_scratch.data_ptr()), ctypes.c_void_p(vis.data_ptr()), f0, nf,
                                         1 if accumulate else 0, _stream_handle(stream)), "xc_fx_channels")
        return vis

    def correlate_host_i4(self, x4_host, vis_host, in4_dev, vis_dev, stream=None):
        """End to end with HOST buffers for 4-bit samples (uint8 [T][F][N][2])."""
        self._check(lib().xc_correlate_host_i4(
            self._h, ctypes.c_void_p(x4_host.data_ptr()), ctypes.c_void_p(vis_host.data_ptr()),
            ctypes.c_void_p(in4_dev.data_ptr()), ctypes.c_void_p(vis_dev.data_ptr()), _stream_handle(stream)),
            "xc_correlate_host_i4")
        return vis_host

    def correlate_host(self, x_host, vis_host, in_dev, vis_dev, stream=None):
        """End to end with HOST buffers (H2D copy, X-engine, D2H copy, stream sync).  in_dev: device scratch of at least
        scratch_in_bytes (new_scratch())."""
        if in_dev.numel() * in_dev.element_size() < self.scratch_in_bytes:
            raise ValueError("in_dev scratch smaller than scratch_in_bytes")
        self._check(lib().xc_correlate_host(
            self._h, ctypes.c_void_p(x_host.data_ptr()), ctypes.c_void_p(vis_host.data_ptr()),
            ctypes.c_void_p(in_dev.data_ptr()), ctypes.c_void_p(vis_dev.data_ptr()), _stream_handle(stream)),
            "xc_correlate_host")
        return vis_host
