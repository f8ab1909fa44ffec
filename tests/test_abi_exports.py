"""CPU-only: the C-ABI library builds, loads and exports every symbol include/asynclane.h declares
(no compute calls here -- there is no GPU in the build container)."""
import ctypes
import os
import re

from paper_2606_08411_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "asynclane.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(al_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_three_hot_calls():
    syms = declared_symbols()
    for name in ("al_lane_attention", "al_kv_refresh", "al_confidence_select", "al_create", "al_destroy"):
        assert name in syms


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in asynclane.h but not exported"
    assert sorted(binding.EXPORTS) == declared_symbols()
    lib.al_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.al_version()


def test_lane_desc_and_shape_struct_layouts():
    assert ctypes.sizeof(binding.al_attn_shape) == 32
    # al_lane_desc is six int32 (24 bytes); workloads emits int32 [n, 6] rows in the same order
    from paper_2606_08411_b200 import workloads as W
    assert W.make_lanes([dict(kv_base_row=3, prefix_len=5, q_lens=[2])]).tolist() == [[0, 3, 5, 0, 2, 0]]


def test_workspace_queries_need_no_gpu():
    lib = binding.load_library()
    # the cluster/DSMEM merge keeps no partials in HBM: confidence_select needs no workspace at all
    assert lib.al_confidence_select_workspace_bytes(0, 100) == 0
    assert lib.al_confidence_select_workspace_bytes(4, 126464) == 0
    shape = binding.Handle.make_shape(28, 4, 128, binding.AL_BF16, 2048)
    assert lib.al_lane_attention_workspace_bytes(ctypes.byref(shape), 8, 256, 1024) > 0


def test_host_step_struct_matches_the_header():
    """al_host_step mirrors the C struct: 25 pointer/int fields, then n_layers, reserved, cache_layer_stride."""
    names = [f[0] for f in binding.al_host_step._fields_]
    assert names[-3:] == ["n_layers", "reserved", "cache_layer_stride"]
    text = open(os.path.join(ROOT, "include", "asynclane.h")).read()
    body = text[text.index("typedef struct {\n  const void* q;"):text.index("} al_host_step;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    declared = re.findall(r"\b([a-z_0-9]+)\s*[;,]", body)
    assert declared == names
