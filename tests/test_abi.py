"""The C-ABI library loads on a CPU-only box, exports every symbol include/*.h declares, and fails
loudly (no fallback) when there is no GPU.  No compute calls here."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tc():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2606_19271_b200 as tc
    return tc


def test_header_symbols_exported(tc):
    header = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include"))))
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(ts_[a-z_0-9]+)\s*\(", header)))
    assert len(declared) >= 20
    assert sorted(tc.EXPORTED_SYMBOLS) == declared
    for name in declared:
        assert hasattr(tc.lib, name), f"{name} declared in turbochunk.h but not exported"


def test_layout_helpers_and_strerror(tc):
    from paper_2606_19271_b200.binding import ts_pool_config
    cfg = ts_pool_config()
    cfg.n_layers, cfg.n_heads, cfg.head_dim, cfg.page_tokens = 40, 40, 128, 256
    cfg.n_pages, cfg.frame_tokens, cfg.window_frames, cfg.max_sessions = 520, 1560, 21, 8
    assert tc.lib.ts_pool_page_bytes(C.byref(cfg)) == 40 * 2 * 40 * 256 * 128 * 2
    assert tc.lib.ts_pool_slab_bytes(C.byref(cfg)) == 520 * 40 * 2 * 40 * 256 * 128 * 2
    cfg.head_dim = 96
    assert tc.lib.ts_pool_page_bytes(C.byref(cfg)) == tc.TS_ERR_INVALID
    cfg.head_dim, cfg.page_tokens = 128, 48
    assert tc.lib.ts_pool_slab_bytes(C.byref(cfg)) == tc.TS_ERR_INVALID
    assert tc.lib.ts_strerror(tc.TS_ERR_NO_PAGES) == b"not enough free device pages"
    assert tc.lib.ts_version().startswith(b"turbochunk")


def test_invalid_config_rejected_before_cuda(tc):
    from paper_2606_19271_b200.binding import ts_pool_config
    cfg = ts_pool_config()
    cfg.n_layers, cfg.n_heads, cfg.head_dim, cfg.page_tokens = 1, 2, 64, 16
    cfg.n_pages, cfg.frame_tokens, cfg.window_frames, cfg.max_sessions = 4, 16, 0, 2
    order = (C.c_int32 * 4)(0, 1, 1, 3)                       # not a permutation
    cfg.free_order = C.cast(order, C.POINTER(C.c_int32))
    h = C.c_void_p()
    assert tc.lib.ts_pool_create(C.byref(cfg), C.byref(h)) == tc.TS_ERR_INVALID
    assert tc.lib.ts_pool_create(None, C.byref(h)) == tc.TS_ERR_INVALID
    assert tc.lib.ts_session_open(None, None) == tc.TS_ERR_INVALID
    # the step-plan calls reject null handles before touching CUDA
    assert tc.lib.ts_step_plan_create(None, 1, None, None, 1, C.byref(h)) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_bind(None, 0, None, None, None, None, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_prepare(None, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_run(None, 0, 0, C.c_float(1.0), 0, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_commit(None, 0, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_destroy(None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_step_plan_block_bytes(None) == 0
    assert tc.lib.ts_pool_clock_probe(None, None) == tc.TS_ERR_INVALID and tc.lib.ts_pool_sched_builds(None) == 0
    # the allocation-free attention entry and the cross-process migration calls: null handles are refused before any CUDA call
    assert tc.lib.ts_static_scratch_bytes() == 256 * 1024
    assert tc.lib.ts_chunk_attention_static(None, 0, 0, None, None, None, None, None, None, None, C.c_float(1.0), None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_pool_export(None, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_peer_open(None, None, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_peer_close(None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_session_freeze(None, 0, None, None, 0) == tc.TS_ERR_INVALID
    assert tc.lib.ts_session_unfreeze(None, 0) == tc.TS_ERR_INVALID
    assert tc.lib.ts_session_import(None, None, None, None, None) == tc.TS_ERR_INVALID
    assert tc.lib.ts_session_release(None, 0, None) == tc.TS_ERR_INVALID
    from paper_2606_19271_b200.binding import ts_migration_ticket_t, ts_pool_export_t
    assert C.sizeof(ts_pool_export_t) == 320 and C.sizeof(ts_migration_ticket_t) == 16      # as include/turbochunk.h declares


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_fails_loudly(tc):
    from paper_2606_19271_b200.binding import ts_pool_config
    cfg = ts_pool_config()
    cfg.n_layers, cfg.n_heads, cfg.head_dim, cfg.page_tokens = 1, 2, 64, 16
    cfg.n_pages, cfg.frame_tokens, cfg.window_frames, cfg.max_sessions = 4, 16, 0, 2
    h = C.c_void_p()
    assert tc.lib.ts_pool_create(C.byref(cfg), C.byref(h)) == tc.TS_ERR_CUDA
    assert not h.value
    assert len(tc.lib.ts_last_cuda_error()) > 0


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_19271_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith(".py"):
                assert "paper_2606_19271_b200" not in open(os.path.join(dirpath, f)).read().replace(
                    "`paper_2606_19271_b200/`", ""), f


def test_headers_are_plain_c(tmp_path):
    """The boundary is a C ABI: both headers compile as C99 on their own (no C++ types, no torch types)."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("gcc not available")
    src = tmp_path / "hdr.c"
    src.write_text('#include "turbochunk.h"\n#include "turbochunk_sched.h"\n'
                   "int main(void) { ts_pool_config c; ts_sched_config s; (void)c; (void)s; return 0; }\n")
    res = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only",
                          "-I", os.path.join(ROOT, "include"), str(src)], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
