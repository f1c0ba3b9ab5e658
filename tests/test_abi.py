"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/gdn.h
declares, mirrors the config struct, and validates arguments.  No compute calls (no GPU here)."""
import ctypes
import re
from pathlib import Path

import pytest

import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import build as gdn_build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module", autouse=True)
def built():
    gdn_build.build()


def header_functions():
    text = (ROOT / "include" / "gdn.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gdn_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = header_functions()
    assert {"gdn_plan", "gdn_forward_chunk", "gdn_destroy"} <= set(names)
    L = gdn.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/gdn.h but not exported"
    assert sorted(gdn.EXPORTED_SYMBOLS) == names


def test_library_has_no_torch_or_python_dependency():
    import subprocess
    out = subprocess.run(["ldd", str(gdn.LIB_PATH)], capture_output=True, text=True).stdout
    assert "torch" not in out and "python" not in out


def test_config_struct_layout_matches_header():
    # 4 + 8*4 + 2*4 + 4 = 48 bytes of 32-bit fields, then four int64 strides
    assert ctypes.sizeof(gdn.GdnConfig) == 48 + 32
    assert gdn.GdnConfig.q_token_stride.offset == 48


def test_version_and_status_strings():
    assert gdn.gdn_version().count(".") == 2
    assert gdn.gdn_status_string(0) == "GDN_OK"
    assert gdn.gdn_status_string(5) == "GDN_ERR_ARCH"


def _cfg(**kw):
    base = dict(B=1, H=2, T=256, d_k=64, d_v=64)
    base.update(kw)
    return gdn.make_config(**base)


@pytest.mark.parametrize("kw,status", [
    (dict(T=100, group=64), gdn.GDN_ERR_INVALID_ARG),            # T % G != 0
    (dict(B=-1), gdn.GDN_ERR_INVALID_ARG),
    (dict(group=0), gdn.GDN_ERR_INVALID_ARG),
    (dict(chunk=96), gdn.GDN_ERR_INVALID_ARG),
    (dict(io_dtype=7), gdn.GDN_ERR_INVALID_ARG),
    (dict(flags=1 << 20), gdn.GDN_ERR_INVALID_ARG),
    (dict(d_k=112), gdn.GDN_ERR_UNSUPPORTED),                     # d_k = 112 with d_v = 64: rectangular 112 is not supported (112 x 112 bf16 is)
    (dict(d_v=48), gdn.GDN_ERR_UNSUPPORTED),
    (dict(flags=gdn.GDN_FLAG_BIDIR), gdn.GDN_ERR_UNSUPPORTED),
    (dict(q_token_stride=3 * 2 * 64 + 4), gdn.GDN_ERR_ALIGNMENT),  # not a multiple of 8
    (dict(k_token_stride=64), gdn.GDN_ERR_INVALID_ARG),            # smaller than H*d
])
def test_plan_validation(kw, status):
    with pytest.raises(gdn.GdnError) as ei:
        gdn.gdn_plan(_cfg(**kw))
    assert ei.value.status == status
    assert gdn.gdn_last_error(None)


def test_struct_size_is_checked():
    cfg = _cfg()
    cfg.struct_size = 12
    with pytest.raises(gdn.GdnError) as ei:
        gdn.gdn_plan(cfg)
    assert ei.value.status == gdn.GDN_ERR_INVALID_ARG


def test_null_arguments():
    L = gdn.lib()
    assert L.gdn_plan(None, None) == gdn.GDN_ERR_INVALID_ARG
    assert L.gdn_destroy(None) == gdn.GDN_OK
    assert L.gdn_forward_chunk(None, None, None, None, None, None, None, None, None, None) == gdn.GDN_ERR_INVALID_ARG


def test_plan_info_and_packed_strides_accepted():
    # packed qkv [B,T,3,H,d]: token stride 3*H*d
    p = gdn.GdnPlan(B=1, H=2, T=128, d_k=64, d_v=64, q_token_stride=3 * 2 * 64, k_token_stride=3 * 2 * 64,
                    v_token_stride=3 * 2 * 64)
    info = p.info
    assert info.path in gdn.PATH_NAMES and info.launches_per_call >= 1
    p.close()


def test_no_device_means_loud_failure_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    p = gdn.GdnPlan(B=1, H=1, T=64, d_k=32, d_v=32, io_dtype=gdn.GDN_FP32)
    L = gdn.lib()
    buf = (ctypes.c_float * 4096)()
    addr = (ctypes.addressof(buf) + 15) & ~15
    st = L.gdn_forward_chunk(p.handle, addr, addr, addr, addr, addr, None, addr + 64, addr, None)
    assert st in (gdn.GDN_ERR_CUDA, gdn.GDN_ERR_ARCH)
    assert gdn.gdn_last_error(p.handle)
    p.close()
