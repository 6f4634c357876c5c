"""CPU checks of the boundary: the library builds, loads, and exports every symbol include/darts.h declares;
host-only entry points validate their arguments (no compute calls without a GPU)."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "darts.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(darts_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols()
    for name in ("darts_prefill", "darts_decode_step", "darts_select_and_compact", "darts_rollout"):
        assert name in syms


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2605_30859_b200 import build
    lib = C.CDLL(build.build())
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_workspace_sizing_and_argument_validation_on_host():
    from paper_2605_30859_b200 import api, workloads as wl
    cfg = wl.CONFIGS["c3"]["model"]
    m = api.model_desc(cfg)
    rt = api.RuntimeDesc(page_size=64, n_pages=20000, max_rows=512, max_prompts=32, max_prompt_len=512, max_new=8192)
    need = C.c_size_t()
    assert api.darts_workspace_bytes(C.byref(m), C.byref(rt), C.byref(need)) == api.OK
    kv = 36 * 20000 * 2 * 8 * 64 * 128 * 2
    assert kv < need.value < kv + (8 << 30)
    rt.page_size = 0
    assert api.darts_workspace_bytes(C.byref(m), C.byref(rt), C.byref(need)) == api.ERR_INVALID_ARG
    rt.page_size = 64
    m.head_dim = 96
    assert api.darts_workspace_bytes(C.byref(m), C.byref(rt), C.byref(need)) == api.ERR_UNSUPPORTED
    assert api.darts_workspace_bytes(None, C.byref(rt), C.byref(need)) == api.ERR_INVALID_ARG
    assert api.darts_decode_step(None) == api.ERR_INVALID_ARG


def test_binding_structs_match_the_header_layout():
    """sizeof of the ctypes mirrors equals what the C compiler lays out for include/darts.h."""
    import subprocess, tempfile
    from paper_2605_30859_b200 import api
    prog = '#include <stdio.h>\n#include "darts.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu\\n", sizeof(darts_model_desc),' \
           'sizeof(darts_weights), sizeof(darts_runtime_desc), sizeof(darts_policy), sizeof(darts_results), sizeof(darts_counters));}'
    with tempfile.TemporaryDirectory() as td:
        open(os.path.join(td, "t.c"), "w").write(prog)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), os.path.join(td, "t.c"), "-o", os.path.join(td, "t")])
        sizes = [int(v) for v in subprocess.check_output([os.path.join(td, "t")]).split()]
    mirrors = [api.ModelDesc, api.Weights, api.RuntimeDesc, api.Policy, api.Results, api.Counters]
    assert sizes == [C.sizeof(t) for t in mirrors]
