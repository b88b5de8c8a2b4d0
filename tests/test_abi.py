"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol
include/caee.h declares, the ctypes structs match the header's layout, and argument
validation answers with error codes (never a crash, never a silent CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_29982_b200 import build
    build.build()
    from paper_2606_29982_b200 import binding
    return binding


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "caee.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(caee_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(B):
    names = _declared_functions()
    assert len(names) >= 15 and set(names) == set(B.EXPORTS)
    lib = C.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert "sm_100a" in B.caee_version()


def test_struct_layouts_match_header(B):
    assert C.sizeof(B.caee_layer_desc) == 16 * 4
    assert C.sizeof(B.caee_prune_params) == 24
    assert C.sizeof(B.caee_expert_weights) == 6 * 8 and C.sizeof(B.caee_prune_out) == 12 * 8
    assert C.sizeof(B.caee_fwd_stats) == 6 * 8 + 4 * 4 + 64 * 8
    assert C.sizeof(B.caee_calib_opts) == 32 and C.sizeof(B.caee_cost_fit) == 40


def _desc(B, **kw):
    d = dict(H=256, I=512, E=8, S=0, k=2, n_group=1, topk_group=1, score_fn=0, norm_topk=1, routed_scale=1.0,
             act_dtype=0, w_dtype=0, D=2, max_tokens=16, expert_kernel=0, device=-1)
    d.update(kw)
    return B.caee_layer_desc(**d)


@pytest.mark.parametrize("kw,code", [(dict(k=9), -1), (dict(E=0), -1), (dict(n_group=3), -1), (dict(topk_group=2), -1),
                                     (dict(H=100), -2), (dict(act_dtype=2), -3), (dict(w_dtype=7), -3), (dict(D=0), -1),
                                     (dict(max_tokens=0), -1), (dict(score_fn=5), -1), (dict(expert_kernel=9), -1),
                                     (dict(E=8, n_group=4, topk_group=1, k=3), -1)])
def test_create_rejects_bad_descriptors(B, kw, code):
    with pytest.raises(B.CaeeError) as ei:
        B.caee_create(_desc(B, **kw))
    assert ei.value.code == code and len(str(ei.value)) > 20


def test_no_cpu_fallback(B):
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.CaeeError) as ei:
        B.caee_create(_desc(B))
    assert ei.value.code == B.CAEE_EUNSUPPORTED and "no CPU fallback" in str(ei.value)


def test_null_context_is_an_error_not_a_crash(B):
    lib = C.CDLL(B.LIB_PATH)
    lib.caee_destroy.argtypes = [C.c_void_p]
    assert lib.caee_destroy(None) == B.CAEE_EINVAL
    lib.caee_moe_forward.argtypes = [C.c_void_p] * 2 + [C.c_int32] + [C.c_void_p] * 4
    assert lib.caee_moe_forward(None, None, 1, None, None, None, None) == B.CAEE_EINVAL
    lib.caee_create.argtypes = [C.c_void_p, C.c_void_p]
    assert lib.caee_create(None, None) == B.CAEE_EINVAL


def test_cache_abi_argument_errors(B):
    """caee_cache_* reject bad arguments without a GPU; an empty cache reports empty slots."""
    lib = C.CDLL(B.LIB_PATH)
    lib.caee_cache_create.argtypes = [C.c_int32, C.c_void_p]
    assert lib.caee_cache_create(4, None) == B.CAEE_EINVAL
    for bad in (0, -3):
        with pytest.raises(B.CaeeError) as ei:
            B.caee_cache_create(bad)
        assert ei.value.code == B.CAEE_EINVAL
    lib.caee_cache_attach.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
    assert lib.caee_cache_attach(None, None, 0) == B.CAEE_EINVAL
    lib.caee_cache_read_stats.argtypes = [C.c_void_p, C.c_void_p]
    assert lib.caee_cache_read_stats(None, None) == B.CAEE_EINVAL
    cache = B.caee_cache_create(5)
    try:
        assert B.caee_cache_snapshot(cache, 5) == [None] * 5
        st = B.caee_cache_read_stats(cache)
        assert (st.hits, st.misses, st.evictions, st.h2d_bytes) == (0, 0, 0, 0)
    finally:
        B.caee_cache_destroy(cache)
    lib.caee_cache_destroy.argtypes = [C.c_void_p]
    lib.caee_cache_destroy.restype = None
    lib.caee_cache_destroy(None)          # a no-op, not a crash


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import, load or link it."""
    pkg = os.path.join(ROOT, "paper_2606_29982_b200")
    bad = re.compile(r"(import\s+oracle|from\s+oracle|from\s+\.\.?oracle|caee_oracle|libcaee_oracle|oracle/|oracle\.py)")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not bad.search(open(os.path.join(dirpath, f)).read()), f
