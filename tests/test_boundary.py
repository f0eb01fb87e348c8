"""Host-side checks of the C-ABI boundary that need no GPU: the library builds, loads, exports every symbol
include/qld.h declares, validates arguments, and refuses to run without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1511_03390_b200 import build, qld
    build.build()
    return qld.load_library()


def test_header_symbols_are_exported(lib):
    from paper_1511_03390_b200 import qld
    header = open(os.path.join(ROOT, "include", "qld.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(qld_[a-z0-9_]+)\s*\(", header))
    assert declared == set(qld.EXPORTS), declared ^ set(qld.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def _cfg(qld, **kw):
    refs = qld.make_refs(kw.pop("refs", [{"nu": 0.1}]))
    cfg = qld.qld_config()
    cfg.H, cfg.W, cfg.dtype, cfg.N, cfg.K = kw.pop("H", 8), kw.pop("W", 8), kw.pop("dtype", 1), kw.pop("N", 16), len(refs)
    cfg.refs = C.cast(refs, C.POINTER(qld.qld_ref))
    for k, v in kw.items():
        setattr(cfg, k, v)
    cfg._keep = refs
    return cfg


def test_argument_validation_without_gpu(lib):
    from paper_1511_03390_b200 import qld
    n = C.c_size_t()
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld)), C.byref(n)) == qld.QLD_OK and n.value > 16 * 8 * 8 * 2
    for bad in (dict(H=0), dict(N=0), dict(dtype=7), dict(refs=[{"nu": 0.5}]), dict(refs=[{"nu": 0.0}]),
                dict(refs=[{"num": 3, "den": 4}]), dict(ring_frames=16), dict(ring_frames=-2), dict(accum=9),
                dict(norm=3), dict(maps=64), dict(refs=[{"nu": 0.1}] * 9)):
        assert lib.qld_workspace_bytes(C.byref(_cfg(qld, **bad)), C.byref(n)) == qld.QLD_E_INVAL, bad
        assert lib.qld_last_error(None) != b""
    # INT_BINS needs rational references and must fit int32
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, accum=qld.QLD_ACC_INT_BINS)), C.byref(n)) == qld.QLD_E_UNSUPPORTED
    big = _cfg(qld, refs=[{"num": 1, "den": 4}], N=200000, accum=qld.QLD_ACC_INT_BINS)
    assert lib.qld_workspace_bytes(C.byref(big), C.byref(n)) == qld.QLD_E_UNSUPPORTED
    # caller-supplied tables lift the nu check (reading G18) but not on rings / integer bins
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, refs=[{"nu": 0.5}], ref_tables_supplied=1)), C.byref(n)) == qld.QLD_OK
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, refs=[{"nu": 0.0}], ref_tables_supplied=1)), C.byref(n)) == qld.QLD_OK
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, ref_tables_supplied=1, ring_frames=40)), C.byref(n)) == qld.QLD_E_UNSUPPORTED
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, ref_tables_supplied=1, accum=qld.QLD_ACC_INT_BINS)), C.byref(n)) == qld.QLD_E_UNSUPPORTED
    assert lib.qld_workspace_bytes(C.byref(_cfg(qld, ref_tables_supplied=2)), C.byref(n)) == qld.QLD_E_INVAL
    assert lib.qld_set_ref_tables(None, 0, None, None, 0) == qld.QLD_E_INVAL and lib.qld_debug_set_tile(None, 0, 0, 0, 0) == qld.QLD_E_INVAL
    ok = _cfg(qld, refs=[{"num": 1, "den": 4}], N=200000, accum=qld.QLD_ACC_INT_BINS, max_value=4095)
    assert lib.qld_workspace_bytes(C.byref(ok), C.byref(n)) == qld.QLD_OK


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1511_03390_b200 import qld
    ctx = C.c_void_p()
    assert lib.qld_create(C.byref(_cfg(qld)), C.byref(ctx)) == qld.QLD_E_CUDA and not ctx.value
    assert b"no CPU fallback" in lib.qld_last_error(None)
    with pytest.raises(qld.QLDError):
        qld.QLD(8, 8, "u16", 16, [{"nu": 0.1}])
    # NULL contexts are rejected, never dereferenced
    assert lib.qld_demod(None, 0, 0) == qld.QLD_E_INVAL and lib.qld_sync(None) == qld.QLD_E_INVAL
    lib.qld_destroy(None)
