"""CPU checks of the boundary: libuniboost.so builds for sm_100a without a GPU, loads, and exports every symbol
that include/uniboost.h declares; the Python structs match the C layout.  No compute calls here."""
import ctypes
import os
import re

from paper_2606_18431_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    lib = ctypes.CDLL(path)
    hdr = open(os.path.join(ROOT, "include", "uniboost.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)          # drop comments
    declared = set(re.findall(r"\b(ub_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations found"
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), f"{name} is declared in uniboost.h but not exported"


def test_struct_layouts_match_the_header():
    assert ctypes.sizeof(binding.UbConfig) == 16 * 4 + 3 * 8 + 4 + 4 + 8
    assert binding.UbConfig.stream.offset == 96
    assert ctypes.sizeof(binding.UbReplica) == 24
    assert binding.UbReplica.hysteresis_us.offset == 8 and binding.UbReplica.gamma.offset == 16
    assert ctypes.sizeof(binding.UbReplicaStats) == 14 * 8 + 9 * 8 + 4 * 8 + 9 * 8 + 4 * 8


def test_error_strings_and_argument_checks_without_a_gpu():
    L = binding.lib()
    assert L.ub_strerror(0) == b"ok"
    assert b"order" in L.ub_strerror(binding.UB_ESTATE)
    h = ctypes.c_void_p()
    assert L.ub_create(None, ctypes.byref(h)) == binding.UB_EINVAL
    cfg = binding.make_config(dict(n_replicas=1, n_traces=1, max_requests=4, queue_cap=4, kv_blocks=8, block_tokens=16,
                                   max_batch=4, chunk_tokens=8, token_budget=8, bin_tokens=256, tok_us=5000))
    cfg.abi_version = 99
    assert L.ub_create(ctypes.byref(cfg), ctypes.byref(h)) == binding.UB_EINVAL
    cfg.abi_version = binding.UB_ABI_VERSION
    cfg.queue_cap = binding.UB_MAX_QUEUE + 1
    assert L.ub_create(ctypes.byref(cfg), ctypes.byref(h)) == binding.UB_EINVAL


def test_product_path_does_not_touch_the_oracle():
    """The CUDA package never imports, links or reads anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2606_18431_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "orc_" not in src and "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libuniboost" not in src and "binding" not in src and "ub_create" not in src, f
