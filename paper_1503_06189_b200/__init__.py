"""Python binding of libxcorr.so -- argument marshalling only; every step of the path runs in the CUDA kernels.

The functions mirror include/xcorr.h one to one (same names, raw pointers as ints).  ``XCorr`` and
``XCorrStream`` are thin conveniences that accept torch tensors (PyTorch is used for device / pinned memory and
stream handles only).  There is no fallback: if the shared library is missing and cannot be built, or the device
is not an sm_100 GPU, the calls raise.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

from . import _build

__all__ = [
    "XCORR_OK", "XCORR_EINVAL", "XCORR_EARCH", "XCORR_ENOMEM", "XCORR_ECUDA", "XCORR_EOVERFLOW", "XCORR_ELIMIT",
    "XCORR_ASSEMBLE_STATIC_MAX_POSITIONS", "xcorr_assemble_static", "xcorr_assemble_static_last_cuda_error",
    "XCorrError", "lib", "xcorr_create", "xcorr_process", "xcorr_read", "xcorr_destroy", "xcorr_strerror",
    "xcorr_last_cuda_error", "xcorr_frame_bytes", "xcorr_output_bytes", "xcorr_kernel_launches",
    "xcorr_norm_enable", "xcorr_norm_process", "xcorr_read_normalized", "xcorr_promise_complete_frames",
    "xcorr_stream_create", "xcorr_stream_submit", "xcorr_stream_sync", "xcorr_stream_read", "xcorr_stream_read_async", "xcorr_stream_destroy",
    "xcorr_assembler_create", "xcorr_assembler_packet_bytes", "xcorr_assemble", "xcorr_assembler_kernel_launches",
    "xcorr_assembler_destroy", "xcorr_norm_process_dev", "xcorr_assemble_accounted", "xcorr_stream_attach_assembler", "xcorr_stream_submit_packets",
    "xcorr_stream_read_normalized",
    "xcorr_debug_schedule", "xcorr_debug_stage_samples", "XCorr", "XCorrStream", "Assembler",
]

XCORR_OK, XCORR_EINVAL, XCORR_EARCH, XCORR_ENOMEM, XCORR_ECUDA, XCORR_EOVERFLOW, XCORR_ELIMIT = 0, -1, -2, -3, -4, -5, -6
XCORR_ASSEMBLE_STATIC_MAX_POSITIONS = 131072   # include/xcorr_assemble.h

_lib = None


class XCorrError(RuntimeError):
    def __init__(self, code: int, what: str, cuda_error: int = 0):
        self.code = code
        self.cuda_error = cuda_error
        msg = f"{what}: {xcorr_strerror(code)} (code {code})"
        if cuda_error:
            msg += f" [cudaError {cuda_error}]"
        super().__init__(msg)


def lib() -> ctypes.CDLL:
    """Load (building first if the sources are newer) libxcorr.so.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path: Path = _build.LIB
    if _build.needs_build():
        try:
            _build.build()
        except Exception as e:  # no nvcc on this box
            if not path.exists():
                raise RuntimeError(f"libxcorr.so is missing and could not be built: {e}") from e
    L = ctypes.CDLL(str(path))
    vp, ci = ctypes.c_void_p, ctypes.c_int
    L.xcorr_create.argtypes = [ci, ci, ci, ctypes.POINTER(vp)]
    L.xcorr_create.restype = ci
    L.xcorr_process.argtypes = [vp, vp, vp]
    L.xcorr_process.restype = ci
    L.xcorr_read.argtypes = [vp, vp, vp]
    L.xcorr_read.restype = ci
    L.xcorr_destroy.argtypes = [vp]
    L.xcorr_destroy.restype = None
    L.xcorr_strerror.argtypes = [ci]
    L.xcorr_strerror.restype = ctypes.c_char_p
    L.xcorr_last_cuda_error.argtypes = [vp]
    L.xcorr_last_cuda_error.restype = ci
    L.xcorr_frame_bytes.argtypes = [vp]
    L.xcorr_frame_bytes.restype = ctypes.c_size_t
    L.xcorr_output_bytes.argtypes = [vp]
    L.xcorr_output_bytes.restype = ctypes.c_size_t
    L.xcorr_kernel_launches.argtypes = [vp]
    L.xcorr_kernel_launches.restype = ctypes.c_uint64
    L.xcorr_promise_complete_frames.argtypes = [vp, ci]
    L.xcorr_promise_complete_frames.restype = ci
    L.xcorr_norm_enable.argtypes = [vp]
    L.xcorr_norm_enable.restype = ci
    L.xcorr_norm_process.argtypes = [vp, vp, vp, vp]
    L.xcorr_norm_process.restype = ci
    L.xcorr_read_normalized.argtypes = [vp, vp, vp, vp]
    L.xcorr_read_normalized.restype = ci
    L.xcorr_stream_create.argtypes = [vp, ci, ctypes.POINTER(vp)]
    L.xcorr_stream_create.restype = ci
    L.xcorr_stream_submit.argtypes = [vp, vp]
    L.xcorr_stream_submit.restype = ci
    L.xcorr_stream_sync.argtypes = [vp]
    L.xcorr_stream_sync.restype = ci
    L.xcorr_stream_read.argtypes = [vp, vp]
    L.xcorr_stream_read.restype = ci
    L.xcorr_stream_read_async.argtypes = [vp, vp]
    L.xcorr_stream_read_async.restype = ci
    L.xcorr_stream_destroy.argtypes = [vp]
    L.xcorr_stream_destroy.restype = None
    L.xcorr_assembler_create.argtypes = [ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
    L.xcorr_assembler_create.restype = ci
    L.xcorr_assembler_packet_bytes.argtypes = [vp]
    L.xcorr_assembler_packet_bytes.restype = ctypes.c_size_t
    L.xcorr_assemble.argtypes = [vp, vp, ctypes.c_size_t, ctypes.c_uint64, vp, vp, vp, vp, vp]
    L.xcorr_assemble.restype = ci
    L.xcorr_assemble_accounted.argtypes = [vp, vp, vp, ctypes.c_size_t, ctypes.c_uint64, vp, vp, vp, vp, vp]
    L.xcorr_assemble_accounted.restype = ci
    L.xcorr_assemble_static.argtypes = [ci, ci, ci, ci, ci, vp, ctypes.c_size_t, ctypes.c_uint64, vp, vp, vp, vp, vp]
    L.xcorr_assemble_static.restype = ci
    L.xcorr_assemble_static_last_cuda_error.argtypes = []
    L.xcorr_assemble_static_last_cuda_error.restype = ci
    L.xcorr_assembler_kernel_launches.argtypes = [vp]
    L.xcorr_assembler_kernel_launches.restype = ctypes.c_uint64
    L.xcorr_assembler_destroy.argtypes = [vp]
    L.xcorr_assembler_destroy.restype = None
    L.xcorr_norm_process_dev.argtypes = [vp, vp, vp, vp]
    L.xcorr_norm_process_dev.restype = ci
    L.xcorr_stream_attach_assembler.argtypes = [vp, vp, ctypes.c_size_t]
    L.xcorr_stream_attach_assembler.restype = ci
    L.xcorr_stream_submit_packets.argtypes = [vp, vp, ctypes.c_size_t, ctypes.c_uint64]
    L.xcorr_stream_submit_packets.restype = ci
    L.xcorr_stream_read_normalized.argtypes = [vp, vp, vp]
    L.xcorr_stream_read_normalized.restype = ci
    L.xcorr_debug_schedule.argtypes = [ci, ci, ci, ci, ctypes.POINTER(ctypes.c_int32), ci, ctypes.POINTER(ctypes.c_int32)]
    L.xcorr_debug_schedule.restype = ci
    L.xcorr_debug_stage_samples.argtypes = []
    L.xcorr_debug_stage_samples.restype = ci
    _lib = L
    return L


# ------------------------------------------------------------------------------------------ raw C-ABI mirrors
def xcorr_strerror(code: int) -> str:
    return lib().xcorr_strerror(int(code)).decode()


def xcorr_create(n_inputs: int, n_freq: int, t_per_frame: int) -> tuple[int, int]:
    """-> (code, handle).  handle is 0 on failure."""
    h = ctypes.c_void_p()
    rc = lib().xcorr_create(int(n_inputs), int(n_freq), int(t_per_frame), ctypes.byref(h))
    return rc, (h.value or 0)


def xcorr_process(handle: int, packed_frame_dev: int, cuda_stream: int = 0) -> int:
    return lib().xcorr_process(handle, packed_frame_dev, cuda_stream)


def xcorr_read(handle: int, upper_triangle_out: int, cuda_stream: int = 0) -> int:
    return lib().xcorr_read(handle, upper_triangle_out, cuda_stream)


def xcorr_destroy(handle: int) -> None:
    lib().xcorr_destroy(handle)


def xcorr_last_cuda_error(handle: int) -> int:
    return lib().xcorr_last_cuda_error(handle)


def xcorr_frame_bytes(handle: int) -> int:
    return lib().xcorr_frame_bytes(handle)


def xcorr_output_bytes(handle: int) -> int:
    return lib().xcorr_output_bytes(handle)


def xcorr_kernel_launches(handle: int) -> int:
    return lib().xcorr_kernel_launches(handle)


def xcorr_promise_complete_frames(handle: int, enabled: int = 1) -> int:
    return lib().xcorr_promise_complete_frames(handle, int(enabled))


def xcorr_norm_enable(handle: int) -> int:
    return lib().xcorr_norm_enable(handle)


def xcorr_norm_process(handle: int, flags_dev: int, lost_samples_host: int, cuda_stream: int = 0) -> int:
    return lib().xcorr_norm_process(handle, flags_dev or None, lost_samples_host or None, cuda_stream)


def xcorr_read_normalized(handle: int, vis_out: int, lost_matrix_out: int = 0, cuda_stream: int = 0) -> int:
    return lib().xcorr_read_normalized(handle, vis_out, lost_matrix_out or None, cuda_stream)


def xcorr_norm_process_dev(handle: int, flags_dev: int, lost_samples_dev: int, cuda_stream: int = 0) -> int:
    return lib().xcorr_norm_process_dev(handle, flags_dev or None, lost_samples_dev or None, cuda_stream)


def xcorr_assembler_create(n_inputs: int, n_freq: int, t_per_frame: int, samples_per_packet: int = 4,
                           freq_per_packet: int = 8) -> tuple[int, int]:
    a = ctypes.c_void_p()
    rc = lib().xcorr_assembler_create(int(n_inputs), int(n_freq), int(t_per_frame), int(samples_per_packet), int(freq_per_packet),
                                      ctypes.byref(a))
    return rc, (a.value or 0)


def xcorr_assembler_packet_bytes(assembler: int) -> int:
    return lib().xcorr_assembler_packet_bytes(assembler)


def xcorr_assemble(assembler: int, packets: int, n_packets: int, seq0: int, frame_dev: int, flags_dev: int = 0, lost_dev: int = 0,
                   counts_dev: int = 0, cuda_stream: int = 0) -> int:
    return lib().xcorr_assemble(assembler, packets or None, int(n_packets), int(seq0), frame_dev or None, flags_dev or None,
                                lost_dev or None, counts_dev or None, cuda_stream)


def xcorr_assemble_accounted(assembler: int, handle: int, packets: int, n_packets: int, seq0: int, frame_dev: int, flags_dev: int = 0,
                             lost_dev: int = 0, counts_dev: int = 0, cuda_stream: int = 0) -> int:
    return lib().xcorr_assemble_accounted(assembler, handle, packets or None, int(n_packets), int(seq0), frame_dev or None,
                                          flags_dev or None, lost_dev or None, counts_dev or None, cuda_stream)


def xcorr_assemble_static(n_inputs: int, n_freq: int, t_per_frame: int, samples_per_packet: int, freq_per_packet: int, packets: int,
                          n_packets: int, seq0: int, frame_dev: int, flags_dev: int = 0, lost_dev: int = 0, counts_dev: int = 0,
                          cuda_stream: int = 0) -> int:
    """xcorr_assemble without an assembler handle and without any allocation: for callers that must not allocate while the
    system runs (per-frame threads of a live acquisition, processes whose device memory another allocator owns).  The
    scratch is a fixed array inside libxcorr.so, so a frame may have at most XCORR_ASSEMBLE_STATIC_MAX_POSITIONS packet
    positions (else XCORR_ELIMIT), and calls that overlap on one GPU race on it.  Make the first call on each device at
    start-up.  Contract: include/xcorr_assemble.h."""
    return lib().xcorr_assemble_static(int(n_inputs), int(n_freq), int(t_per_frame), int(samples_per_packet), int(freq_per_packet),
                                       packets or None, int(n_packets), int(seq0), frame_dev or None, flags_dev or None,
                                       lost_dev or None, counts_dev or None, cuda_stream)


def xcorr_assemble_static_last_cuda_error() -> int:
    return lib().xcorr_assemble_static_last_cuda_error()


def xcorr_assembler_kernel_launches(assembler: int) -> int:
    return lib().xcorr_assembler_kernel_launches(assembler)


def xcorr_assembler_destroy(assembler: int) -> None:
    lib().xcorr_assembler_destroy(assembler)


def xcorr_stream_create(handle: int, depth: int = 2) -> tuple[int, int]:
    s = ctypes.c_void_p()
    rc = lib().xcorr_stream_create(handle, int(depth), ctypes.byref(s))
    return rc, (s.value or 0)


def xcorr_stream_submit(stream: int, frame_host: int) -> int:
    return lib().xcorr_stream_submit(stream, frame_host)


def xcorr_stream_sync(stream: int) -> int:
    return lib().xcorr_stream_sync(stream)


def xcorr_stream_read(stream: int, upper_triangle_out: int) -> int:
    return lib().xcorr_stream_read(stream, upper_triangle_out)


def xcorr_stream_read_async(stream: int, upper_triangle_out: int) -> int:
    return lib().xcorr_stream_read_async(stream, upper_triangle_out)


def xcorr_stream_attach_assembler(stream: int, assembler: int, max_packets: int) -> int:
    return lib().xcorr_stream_attach_assembler(stream, assembler, int(max_packets))


def xcorr_stream_submit_packets(stream: int, packets_host: int, n_packets: int, seq0: int) -> int:
    return lib().xcorr_stream_submit_packets(stream, packets_host or None, int(n_packets), int(seq0))


def xcorr_stream_read_normalized(stream: int, vis_out: int, lost_matrix_out: int = 0) -> int:
    return lib().xcorr_stream_read_normalized(stream, vis_out, lost_matrix_out or None)


def xcorr_stream_destroy(stream: int) -> None:
    lib().xcorr_stream_destroy(stream)


def xcorr_debug_stage_samples() -> int:
    return lib().xcorr_debug_stage_samples()


def xcorr_debug_schedule(n_inputs: int, n_freq: int, t_per_frame: int, n_workers: int):
    """-> (segments int32[K][7] = f, I, J, stage_begin, stage_end, tile, slot ; worker_begin int32[n_workers+1]).  No GPU needed."""
    import numpy as np
    n = lib().xcorr_debug_schedule(n_inputs, n_freq, t_per_frame, n_workers, None, 0, None)
    if n < 0:
        raise XCorrError(n, "xcorr_debug_schedule")
    seg = np.zeros((max(n, 1), 7), dtype=np.int32)
    wb = np.zeros(n_workers + 1, dtype=np.int32)
    n2 = lib().xcorr_debug_schedule(n_inputs, n_freq, t_per_frame, n_workers,
                                    seg.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), n,
                                    wb.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)))
    assert n2 == n
    return seg[:n], wb


# ------------------------------------------------------------------------------------------ torch conveniences
def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class XCorr:
    """One (N, F, T) correlator handle.  ``process`` accumulates a device frame, ``read`` ends the integration."""

    def __init__(self, n_inputs: int, n_freq: int, t_per_frame: int):
        rc, h = xcorr_create(n_inputs, n_freq, t_per_frame)
        if rc != XCORR_OK:
            raise XCorrError(rc, "xcorr_create")
        self.handle = h
        self.n_inputs, self.n_freq, self.t_per_frame = n_inputs, n_freq, t_per_frame
        self.n_pairs = n_inputs * (n_inputs + 1) // 2

    @property
    def frame_bytes(self) -> int:
        return xcorr_frame_bytes(self.handle)

    @property
    def output_bytes(self) -> int:
        return xcorr_output_bytes(self.handle)

    @property
    def kernel_launches(self) -> int:
        return xcorr_kernel_launches(self.handle)

    def _stream(self, stream) -> int:
        """The cudaStream_t of ``stream``; keeps the stream OBJECT referenced until this handle's next call has been given its
        own: the library records an event on the previous call's stream at the next call (stream order, include/xcorr.h),
        so that stream must not be destroyed by Python's garbage collector in between."""
        self._prev_stream, self._last_stream = getattr(self, "_last_stream", None), stream   # the previous one lives through this call
        return _stream_handle(stream)

    def _check(self, rc: int, what: str):
        if rc != XCORR_OK:
            raise XCorrError(rc, what, xcorr_last_cuda_error(self.handle))

    def process(self, frame_dev, stream=None) -> None:
        """frame_dev: torch uint8 CUDA tensor of N*F*T bytes ([T][F][N]), contiguous."""
        if not frame_dev.is_cuda or not frame_dev.is_contiguous() or frame_dev.numel() * frame_dev.element_size() != self.frame_bytes:
            raise ValueError("frame_dev must be a contiguous CUDA tensor of exactly frame_bytes bytes")
        self._check(xcorr_process(self.handle, frame_dev.data_ptr(), self._stream(stream)), "xcorr_process")

    def read(self, out=None, stream=None):
        """Write int32[F][P][2] into ``out`` (CUDA or CPU torch int32 tensor; allocated on the device if None)."""
        import torch
        if out is None:
            out = torch.empty((self.n_freq, self.n_pairs, 2), dtype=torch.int32, device="cuda")
        if out.dtype != torch.int32 or not out.is_contiguous() or out.numel() * 4 != self.output_bytes:
            raise ValueError("out must be a contiguous int32 tensor of output_bytes bytes")
        self._check(xcorr_read(self.handle, out.data_ptr(), self._stream(stream)), "xcorr_read")
        return out

    def promise_complete_frames(self, enabled: bool = True) -> None:
        """See xcorr_promise_complete_frames in include/xcorr.h."""
        self._check(xcorr_promise_complete_frames(self.handle, 1 if enabled else 0), "xcorr_promise_complete_frames")

    # ---- lost-sample normalisation (NEXT-1)
    def norm_enable(self) -> None:
        self._check(xcorr_norm_enable(self.handle), "xcorr_norm_enable")

    def norm_process(self, flags_dev=None, lost_samples=None, stream=None) -> None:
        """flags_dev: CUDA uint8 tensor [T][F][N/8] or None; lost_samples: int32 numpy array [F] (host) or None."""
        import numpy as np
        fptr = 0
        if flags_dev is not None:
            if not flags_dev.is_cuda or not flags_dev.is_contiguous() or flags_dev.numel() * flags_dev.element_size() * 8 != self.frame_bytes:
                raise ValueError("flags_dev must be a contiguous CUDA tensor of frame_bytes / 8 bytes")
            fptr = flags_dev.data_ptr()
        lptr = 0
        if lost_samples is not None:
            lost_samples = np.ascontiguousarray(lost_samples, dtype=np.int32)
            if lost_samples.shape != (self.n_freq,):
                raise ValueError("lost_samples must have shape (n_freq,)")
            lptr = lost_samples.ctypes.data
        self._check(xcorr_norm_process(self.handle, fptr, lptr, self._stream(stream)), "xcorr_norm_process")

    def norm_process_dev(self, flags_dev=None, lost_dev=None, stream=None) -> None:
        """As norm_process with the packet-loss counters in a CUDA int32 tensor [F] (the output of Assembler.assemble)."""
        fptr = flags_dev.data_ptr() if flags_dev is not None else 0
        if flags_dev is not None and (not flags_dev.is_cuda or flags_dev.numel() * flags_dev.element_size() * 8 != self.frame_bytes):
            raise ValueError("flags_dev must be a contiguous CUDA tensor of frame_bytes / 8 bytes")
        if lost_dev is not None and (not lost_dev.is_cuda or lost_dev.numel() != self.n_freq or lost_dev.element_size() != 4):
            raise ValueError("lost_dev must be a CUDA int32 tensor of n_freq elements")
        lptr = lost_dev.data_ptr() if lost_dev is not None else 0
        self._check(xcorr_norm_process_dev(self.handle, fptr, lptr, self._stream(stream)), "xcorr_norm_process_dev")

    def read_normalized(self, out=None, lost_out=None, stream=None):
        """-> float32[F][P][2] (allocated on the device if None); lost_out: optional int32[F][P] tensor for L."""
        import torch
        if out is None:
            out = torch.empty((self.n_freq, self.n_pairs, 2), dtype=torch.float32, device="cuda")
        if out.dtype != torch.float32 or not out.is_contiguous() or out.numel() * 4 != self.output_bytes:
            raise ValueError("out must be a contiguous float32 tensor of output_bytes bytes")
        lptr = 0
        if lost_out is not None:
            if lost_out.dtype != torch.int32 or not lost_out.is_contiguous() or lost_out.numel() * 8 != self.output_bytes:
                raise ValueError("lost_out must be a contiguous int32 tensor of n_freq * n_pairs elements")
            lptr = lost_out.data_ptr()
        self._check(xcorr_read_normalized(self.handle, out.data_ptr(), lptr, self._stream(stream)), "xcorr_read_normalized")
        return out

    def close(self) -> None:
        if getattr(self, "handle", 0):
            xcorr_destroy(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class XCorrStream:
    """Double-buffered pinned-host -> device frame stream over an ``XCorr`` (hot-path row a5)."""

    def __init__(self, xc: XCorr, depth: int = 2):
        rc, s = xcorr_stream_create(xc.handle, depth)
        if rc != XCORR_OK:
            raise XCorrError(rc, "xcorr_stream_create", xcorr_last_cuda_error(xc.handle))
        self.xc, self.stream = xc, s

    def submit(self, frame_host) -> None:
        """frame_host: contiguous CPU uint8 tensor (pinned for overlap) or numpy array of frame_bytes bytes."""
        if hasattr(frame_host, "data_ptr"):
            ptr, nbytes = frame_host.data_ptr(), frame_host.numel() * frame_host.element_size()
        else:
            ptr, nbytes = frame_host.ctypes.data, frame_host.nbytes
        if nbytes != self.xc.frame_bytes:
            raise ValueError("frame_host must hold exactly frame_bytes bytes")
        self.xc._check(xcorr_stream_submit(self.stream, ptr), "xcorr_stream_submit")

    def sync(self) -> None:
        self.xc._check(xcorr_stream_sync(self.stream), "xcorr_stream_sync")

    def read(self, out):
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        self.xc._check(xcorr_stream_read(self.stream, ptr), "xcorr_stream_read")
        return out

    def attach_assembler(self, assembler, max_packets: int) -> None:
        """Packet path: ``assembler`` is an ``Assembler`` of the same shape; keeps a reference to it."""
        self.xc._check(xcorr_stream_attach_assembler(self.stream, assembler.handle, max_packets), "xcorr_stream_attach_assembler")
        self.assembler = assembler

    def submit_packets(self, packets_host, n_packets: int, seq0: int) -> None:
        """packets_host: contiguous (pinned) CPU uint8 tensor / numpy array holding n_packets packets in arrival order."""
        if hasattr(packets_host, "data_ptr"):
            ptr, nbytes = packets_host.data_ptr(), packets_host.numel() * packets_host.element_size()
        else:
            ptr, nbytes = packets_host.ctypes.data, packets_host.nbytes
        if nbytes < n_packets * self.assembler.packet_bytes:
            raise ValueError("packets_host holds fewer than n_packets packets")
        self.xc._check(xcorr_stream_submit_packets(self.stream, ptr, n_packets, seq0), "xcorr_stream_submit_packets")

    def read_normalized(self, out, lost_out=None):
        lptr = 0 if lost_out is None else (lost_out.data_ptr() if hasattr(lost_out, "data_ptr") else lost_out.ctypes.data)
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        self.xc._check(xcorr_stream_read_normalized(self.stream, ptr, lptr), "xcorr_stream_read_normalized")
        return out

    def read_async(self, out):
        """Enqueue the read without waiting; ``out`` is valid after ``sync()``."""
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        self.xc._check(xcorr_stream_read_async(self.stream, ptr), "xcorr_stream_read_async")
        return out

    def close(self) -> None:
        if getattr(self, "stream", 0):
            xcorr_stream_destroy(self.stream)
            self.stream = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Assembler:
    """Packet -> frame assembly (NEXT-2, include/xcorr_assemble.h): packets in arrival order -> frame, flags, loss counters."""

    def __init__(self, n_inputs: int, n_freq: int, t_per_frame: int, samples_per_packet: int = 4, freq_per_packet: int = 8):
        rc, a = xcorr_assembler_create(n_inputs, n_freq, t_per_frame, samples_per_packet, freq_per_packet)
        if rc != XCORR_OK:
            raise XCorrError(rc, "xcorr_assembler_create")
        self.handle = a
        self.n_inputs, self.n_freq, self.t_per_frame = n_inputs, n_freq, t_per_frame
        self.packet_bytes = xcorr_assembler_packet_bytes(a)

    @property
    def kernel_launches(self) -> int:
        return xcorr_assembler_kernel_launches(self.handle)

    def assemble(self, packets, n_packets: int, seq0: int, frame=None, flags=None, lost=None, counts=None, stream=None, account_into=None):
        """packets: CUDA or pinned-CPU uint8 tensor holding >= n_packets packets back to back (arrival order).
        frame / flags / lost / counts: CUDA output tensors (allocated if None; ``flags=False``: no flag field is written and
        None is returned in its place).  -> (frame, flags, lost, counts).
        account_into: an ``XCorr`` with normalisation enabled -> xcorr_assemble_accounted (flags and losses are counted into
        that handle in the same pass; no separate norm_process call is needed)."""
        import torch
        if packets is not None and packets.numel() * packets.element_size() < n_packets * self.packet_bytes:
            raise ValueError("packets holds fewer than n_packets packets")
        if packets is not None and not packets.is_cuda and not packets.is_pinned():
            raise ValueError("host packets must be page-locked (pin_memory) so the GPU can read them")
        t, f, n = self.t_per_frame, self.n_freq, self.n_inputs
        frame = torch.empty((t, f, n), dtype=torch.uint8, device="cuda") if frame is None else frame
        if flags is False:           # no flag field wanted (the C ABI's NULL): what the streamed packet path does when it accounts in-pass
            flags = None
            fptr = 0
        else:
            flags = torch.empty((t, f, n // 8), dtype=torch.uint8, device="cuda") if flags is None else flags
            fptr = flags.data_ptr()
        lost = torch.empty(f, dtype=torch.int32, device="cuda") if lost is None else lost
        counts = torch.empty(4, dtype=torch.int32, device="cuda") if counts is None else counts
        if frame.numel() != t * f * n or (flags is not None and flags.numel() * 8 != t * f * n) or lost.numel() != f or counts.numel() != 4:
            raise ValueError("output tensor of the wrong size")
        pptr = packets.data_ptr() if packets is not None else 0
        if account_into is None:
            rc = xcorr_assemble(self.handle, pptr, n_packets, seq0, frame.data_ptr(), fptr, lost.data_ptr(), counts.data_ptr(),
                                _stream_handle(stream))
        else:
            rc = xcorr_assemble_accounted(self.handle, account_into.handle, pptr, n_packets, seq0, frame.data_ptr(), fptr,
                                          lost.data_ptr(), counts.data_ptr(), account_into._stream(stream))
        if rc != XCORR_OK:
            raise XCorrError(rc, "xcorr_assemble")
        return frame, flags, lost, counts

    def close(self) -> None:
        if getattr(self, "handle", 0):
            xcorr_assembler_destroy(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
