"""The C-ABI library loads and exports every symbol include/*.h declares (no compute calls: CPU only)."""
import ctypes
import re
from pathlib import Path

import pytest

import paper_1503_06189_b200 as xb

INCLUDE = Path(__file__).resolve().parent.parent / "include"


def _declared_symbols():
    names = []
    for h in sorted(INCLUDE.glob("*.h")):
        text = re.sub(r"/\*.*?\*/", "", h.read_text(), flags=re.S)
        for m in re.finditer(r"\b(xcorr_[a-z0-9_]+)\s*\(", text):
            names.append(m.group(1))
    return sorted(set(names))


def test_headers_declare_the_three_calls():
    names = _declared_symbols()
    for must in ("xcorr_create", "xcorr_process", "xcorr_read", "xcorr_destroy", "xcorr_strerror",
                 "xcorr_stream_create", "xcorr_stream_submit", "xcorr_stream_read"):
        assert must in names


@pytest.mark.parametrize("name", _declared_symbols())
def test_symbol_exported(name):
    L = xb.lib()
    assert getattr(L, name) is not None


def test_library_exports_only_the_declared_c_abi():
    """libxcorr.so carries no test scaffolding and no measurement code: every extern "C" symbol it exports is declared in
    include/*.h (the SIMT second opinion lives in tests/support, the int8 issue probe in libxcorr_probe.so)."""
    import subprocess
    from paper_1503_06189_b200 import _build
    xb.lib()
    out = subprocess.run(["nm", "-D", "--defined-only", str(_build.LIB)], capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if ln.split() and not ln.split()[-1].startswith("_")}
    c_abi = {name for name in exported if name.startswith("xcorr_")}
    assert c_abi == set(_declared_symbols())
    assert not any("simt" in name.lower() or "probe" in name.lower() or "profile" in name.lower() for name in exported)


def test_support_libraries_build_and_export():
    """The two non-product libraries build for sm_100a without a GPU and export their one entry point each."""
    from bench_support import probe
    from tests import support
    assert probe.lib().xcorr_probe_int8_issue is not None
    assert support.lib().simt_xcorr is not None


def test_no_torch_types_in_abi():
    for h in INCLUDE.glob("*.h"):
        code = re.sub(r"/\*.*?\*/", "", h.read_text(), flags=re.S)   # comments may mention torch pin_memory
        assert "torch" not in code.lower() and "at::" not in code and "#include <cuda" not in code


def test_strerror_is_total():
    for code in range(-8, 2):
        s = xb.xcorr_strerror(code)
        assert isinstance(s, str) and s
    assert xb.xcorr_strerror(xb.XCORR_OK) == "ok"
    assert "overflow" in xb.xcorr_strerror(xb.XCORR_EOVERFLOW)


@pytest.mark.parametrize("shape", [(0, 4, 16), (16, 0, 16), (16, 4, 0), (-16, 4, 16), (24, 4, 16), (8, 1, 1), (250, 2, 64),
                                   # shapes whose work tables alone would not fit: refused before any schedule is built
                                   (65536, 65535, 16), (65536, 9, 16), (4096, 2049, 16)])
def test_create_rejects_bad_shapes_without_touching_the_gpu(shape):
    rc, h = xb.xcorr_create(*shape)
    assert rc == xb.XCORR_EINVAL and h == 0


def test_schedule_of_an_oversized_shape_is_refused_not_attempted():
    with pytest.raises(xb.XCorrError):
        xb.xcorr_debug_schedule(65536, 65535, 16, 74)
    with pytest.raises(xb.XCorrError):
        xb.xcorr_debug_schedule(4096, 2048, 64, 74)                 # 2048 channels x 136 super-tiles = 278,528 > 2^18 work items
    seg, wb = xb.xcorr_debug_schedule(4096, 1927, 64, 74)           # 262,072 work items: the largest that is still scheduled
    assert len(seg) >= 262072 and wb[-1] == len(seg)


def test_null_handles_are_harmless():
    assert xb.xcorr_frame_bytes(0) == 0
    assert xb.xcorr_output_bytes(0) == 0
    assert xb.xcorr_kernel_launches(0) == 0
    assert xb.xcorr_last_cuda_error(0) == 0
    xb.xcorr_destroy(0)
    xb.xcorr_stream_destroy(0)
    assert xb.xcorr_process(0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_read(0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_stream_submit(0, 0) == xb.XCORR_EINVAL


@pytest.mark.parametrize("args", [(16, 8, 16, 0, 8), (16, 8, 16, 4, 0), (16, 8, 18, 4, 8), (16, 12, 16, 4, 8), (16, 8, 16, 4, 4),
                                  (24, 8, 16, 4, 8)])
def test_assembler_create_rejects_bad_shapes_without_touching_the_gpu(args):
    rc, a = xb.xcorr_assembler_create(*args)
    assert rc == xb.XCORR_EINVAL and a == 0


def test_assembler_null_handles_are_harmless():
    assert xb.xcorr_assembler_packet_bytes(0) == 0
    assert xb.xcorr_assembler_kernel_launches(0) == 0
    xb.xcorr_assembler_destroy(0)
    assert xb.xcorr_assemble(0, 0, 0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_assemble_accounted(0, 0, 0, 0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_norm_process_dev(0, 0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_stream_attach_assembler(0, 0, 16) == xb.XCORR_EINVAL
    assert xb.xcorr_stream_submit_packets(0, 0, 0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_stream_read_normalized(0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_stream_read_async(0, 0) == xb.XCORR_EINVAL
    assert xb.xcorr_promise_complete_frames(0, 1) == xb.XCORR_EINVAL


def test_create_fails_loudly_without_a_gpu():
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("GPU present")
    except ImportError:
        pass
    rc, h = xb.xcorr_create(16, 4, 256)
    assert rc in (xb.XCORR_ECUDA, xb.XCORR_EARCH) and h == 0
    with pytest.raises(xb.XCorrError):
        xb.XCorr(16, 4, 256)
