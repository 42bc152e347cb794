"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports what
include/lpc.h declares; argument validation that happens before any CUDA call."""
import ctypes
import importlib.util
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lpc():
    spec = importlib.util.spec_from_file_location("_lpc_build", os.path.join(ROOT, "paper_2603_22553_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()
    import paper_2603_22553_b200 as m
    return m


def _declared():
    text = open(os.path.join(ROOT, "include", "lpc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lpc_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lpc):
    lib = ctypes.CDLL(lpc.LIB_PATH)
    names = _declared()
    assert {"lpc_create_lattice", "lpc_set_site_params", "lpc_step_n", "lpc_read_fid", "lpc_moments"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(lpc.EXPORTS)


def test_workspace_bytes_and_validation_without_gpu(lpc):
    cfg = lpc.make_config(512, 512, 512, max_steps=1000)
    b = lpc.lpc_workspace_bytes(cfg)
    n = 512 ** 3
    assert 56 * n < b < 63 * n          # 56 B/site algorithmic (h x2 buffers, pi, cos, sin) + ghost padding + series
    cfg5 = lpc.make_config(256, 256, 256, n_moments=3, max_steps=10)
    assert lpc.lpc_workspace_bytes(cfg5) > lpc.lpc_workspace_bytes(lpc.make_config(256, 256, 256, max_steps=10))
    f32 = lpc.lpc_workspace_bytes(lpc.make_config(512, 512, 512, precision=1, max_steps=1000))
    assert f32 < 0.56 * b
    for bad in (dict(nx=0), dict(alpha=0.0), dict(alpha=1.5), dict(n_moments=2), dict(precision=3), dict(dt=0.0),
                dict(max_steps=-1), dict(bc=(0, 2, 0)), dict(n_density=4)):
        kw = dict(nx=8, ny=8, nz=8)
        kw.update(bad)
        with pytest.raises(lpc.LpcError) as ei:
            lpc.lpc_workspace_bytes(lpc.make_config(**kw))
        assert ei.value.code == lpc.LPC_EINVAL
        assert lpc.lpc_last_error() != ""


def test_missing_library_fails_loudly(lpc, monkeypatch):
    import paper_2603_22553_b200 as m
    monkeypatch.setattr(m, "_lib_handle", None)
    monkeypatch.setattr(m, "LIB_PATH", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(ImportError):
        m.lpc_workspace_bytes(m.make_config(4, 4, 4))
