"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/prr.h
declares, validates its arguments before touching CUDA and refuses to run without a device (no
CPU fallback).  No compute calls are made here."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2606_30389_b200 import prr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "prr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(prr_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert len(names) >= 25 and "prr_decode_step" in names and "prr_calibrate" in names
    L = prr.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/prr.h but not exported by libprr.so"
    assert sorted(prr.SYMBOLS) == names, "binding's symbol list is out of sync with include/prr.h"
    assert b"sm_100a" in L.prr_version()


def test_binding_structs_match_header_layout():
    # field order and sizes of the two C structs (10 x 4 bytes; 4 pointers + 2 int32)
    assert C.sizeof(prr.Layout) == 40
    assert C.sizeof(prr.PagedKV) == 4 * C.sizeof(C.c_void_p) + 8
    assert [f[0] for f in prr.Layout._fields_] == [
        "n_q_heads", "n_kv_heads", "head_dim", "max_batch", "max_blocks_per_seq", "n_layers", "kv_dtype",
        "overpredict_policy", "sm_scale", "orchestration"]


@pytest.mark.parametrize("args,code", [
    (dict(n_q_heads=30, n_kv_heads=8), prr.E_INVALID),          # not a multiple
    (dict(head_dim=96), prr.E_UNSUPPORTED),
    (dict(block_size=48), prr.E_UNSUPPORTED),
    (dict(K=0), prr.E_INVALID),
    (dict(budget=-1), prr.E_INVALID),
    (dict(n_q_heads=34, n_kv_heads=2), prr.E_UNSUPPORTED),      # G = 17
    (dict(max_blocks_per_seq=40000), prr.E_UNSUPPORTED),
    (dict(policy=7), prr.E_INVALID),
])
def test_create_validates_before_cuda(args, code):
    kw = dict(n_q_heads=32, n_kv_heads=8, head_dim=128, block_size=64, K=8, budget=8)
    kw.update(args)
    with pytest.raises(prr.PrrError) as e:
        prr.Context(**kw)
    assert e.value.code == code and "prr_create" in str(e.value)


def test_null_arguments_are_invalid_not_crashes():
    L = prr.lib()
    assert L.prr_create(None, 64, 8, 8, None) == prr.E_INVALID
    assert L.prr_destroy(None) == prr.E_INVALID
    assert L.prr_decode_step(None, None, None, None, None, None) == prr.E_INVALID
    assert L.prr_score(None, None, None, None, None, None) == prr.E_INVALID
    assert L.prr_get_stats(None, None, 0, None) == prr.E_INVALID
    assert L.prr_graph_launch(None, None) == prr.E_INVALID
    assert L.prr_launch_count(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback_without_a_device():
    with pytest.raises(prr.PrrError) as e:
        prr.Context(32, 8, 128, 64, 8, 8)
    assert e.value.code == prr.E_CUDA and "no CPU fallback" in str(e.value)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_30389_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle|#\s*include[^\n]*oracle|oracle[/.]prr_oracle|dlopen", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not pat.search(txt), f"{f} reaches into oracle/"
    assert not pat.search(open(os.path.join(ROOT, "include", "prr.h")).read())
