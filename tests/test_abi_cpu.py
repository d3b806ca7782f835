"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every function
include/tts.h declares; the ctypes binding mirrors the header; without a CUDA device the
library fails loudly (no CPU fallback).  No compute calls."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2605_09329_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "tts.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tts_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    assert "tts_distill_step" in names and "tts_accept_mask" in names
    assert len(names) >= 14


def test_library_exports_every_declared_symbol(built):
    lib = ctypes.CDLL(built)
    for name in _declared():
        assert hasattr(lib, name), name


def test_binding_covers_every_declared_symbol(built):
    from paper_2605_09329_b200 import tts
    assert sorted(tts.EXPORTS) == _declared()
    for name in _declared():
        assert callable(getattr(tts, name)), name
    assert tts.tts_version() >= 200
    assert tts.tts_status_string(tts.TTS_ERR_ARCH) == "TTS_ERR_ARCH"


def test_config_struct_matches_header():
    from paper_2605_09329_b200 import tts
    src = open(os.path.join(ROOT, "include", "tts.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} tts_config;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        ty, rest = decl.split(None, 1)
        fields += [(n.strip(), ty) for n in rest.split(",")]
    want = [(n, "int32_t" if t is ctypes.c_int32 else "float") for n, t in tts.tts_config._fields_]
    assert fields == want


def test_enums_match_header():
    from paper_2605_09329_b200 import tts
    from workloads import synth
    src = open(os.path.join(ROOT, "include", "tts.h")).read()
    for m in re.finditer(r"enum\s*\{(.*?)\}", src, flags=re.S):
        body = re.sub(r"/\*.*?\*/", "", m.group(1), flags=re.S)
        nxt = 0
        for item in body.split(","):
            item = item.strip()
            if not item:
                continue
            if "=" in item:
                name, val = [x.strip() for x in item.split("=")]
                nxt = int(val)
            else:
                name = item
            assert getattr(tts, name) == nxt, name
            nxt += 1
    assert (synth.F32, synth.BF16) == (tts.TTS_F32, tts.TTS_BF16)
    assert (synth.SGD, synth.ADAMW) == (tts.TTS_SGD, tts.TTS_ADAMW)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback(built):
    from paper_2605_09329_b200 import tts
    with pytest.raises(tts.TTSError) as e:
        tts.tts_ctx_create(tts.make_config(1024, 64, 8, 8), 0)
    assert e.value.status in (tts.TTS_ERR_CUDA, tts.TTS_ERR_ARCH)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2605_09329_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "tts_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2605_09329_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2605_09329_b200/``", ""), f


def test_unknown_moment_format_is_refused_without_a_gpu(built):
    """The 8-bit moment format was a declared-but-unbuilt enum value (2) up to 0.2.0; it is gone from header and
    binding, and the value is refused by argument checking alone (before any CUDA call)."""
    from paper_2605_09329_b200 import tts
    assert not hasattr(tts, "TTS_MOMENT_Q8") and "TTS_MOMENT_Q8 =" not in open(os.path.join(ROOT, "include", "tts.h")).read()
    with pytest.raises(tts.TTSError) as e:
        tts.tts_ctx_create(tts.make_config(1024, 128, 16, 16, moment_dtype=2), 0)
    assert e.value.status == tts.TTS_ERR_UNSUPPORTED
    assert tts.tts_version() >= 300
