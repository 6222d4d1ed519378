"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/layup.h
declares, its pure host functions agree with the oracle, and without a GPU it fails
loudly instead of falling back (no compute calls here)."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

import oracle
import paper_2410_05985_b200 as pkg
from paper_2410_05985_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_05985_b200.build import build
    build()
    return pkg.load_library()


def test_every_declared_symbol_is_exported(lib):
    text = open(os.path.join(ROOT, "include", "layup.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(layup_[a-z_]+)\s*\(", text))
    assert declared and declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_header_and_binding_structs_agree(lib):
    # the ctypes struct mirrors layup_config field by field
    text = open(os.path.join(ROOT, "include", "layup.h")).read()
    body = re.search(r"typedef struct \{((?:(?!typedef struct).)*?)\} layup_config;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"(\w+)\s*;", body)
    assert names == [f[0] for f in binding._Config._fields_]


def test_tuning_block_is_the_only_switch(lib):
    """layup_tuning (include/layup.h) mirrors the binding field by field, every field is documented
    in the header, and the library reads no environment variable."""
    text = open(os.path.join(ROOT, "include", "layup.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} layup_tuning;", text, flags=re.S).group(1)
    fields = re.findall(r"int32_t\s+(\w+)\s*;\s*/\*", body)               # name followed by its comment
    assert fields == [f[0] for f in binding._Tuning._fields_] and len(fields) == 11
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2410_05985_b200")):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h", ".py")):
                src = open(os.path.join(dirpath, f)).read()
                assert "getenv" not in src and "os.environ" not in src.replace('os.environ.get("CUDA_HOME"', ""), f
    # out-of-range tuning is an argument error, caught before any CUDA call
    arr = (ctypes.c_int64 * 1)(100)
    for bad in (dict(engine=3), dict(launch_shape=-1), dict(fused=5), dict(stages=-2)):
        tune = binding._Tuning(**bad)
        cfg = binding._Config(4, 1, arr, 0.01, 0.0, 0, 0, 0.0, 0, tuning=ctypes.pointer(tune))
        n = ctypes.c_size_t()
        assert lib.layup_arena_bytes(ctypes.byref(cfg), ctypes.byref(n)) == pkg.LAYUP_EINVAL


def test_arena_bytes_layout():
    # slices padded to 32 floats, X|G(|M) sections
    assert pkg.layup_arena_bytes(4, [1, 31, 32, 33], 0.0) == 4 * (32 + 32 + 32 + 64) * 4 * 2
    assert pkg.layup_arena_bytes(4, [1, 31, 32, 33], 0.9) == 4 * (32 + 32 + 32 + 64) * 4 * 3
    assert pkg.layup_arena_bytes(4, [1, 31, 32, 33], 0.0, optimizer=pkg.OPT_ADAMW) == 4 * (32 + 32 + 32 + 64) * 4 * 4
    with pytest.raises(pkg.LayUpError) as e:
        pkg.layup_arena_bytes(0, [10])
    assert e.value.code == pkg.LAYUP_EINVAL
    with pytest.raises(pkg.LayUpError):
        pkg.layup_arena_bytes(4, [10, 0])
    with pytest.raises(pkg.LayUpError):
        pkg.layup_arena_bytes(2000, [10])


def test_host_peer_function_matches_oracle():
    rng = np.random.default_rng(0)
    for _ in range(3000):
        K = int(rng.integers(2, 65))
        seed = int(rng.integers(0, 2**63))
        step = int(rng.integers(0, 2**32))
        layer = int(rng.integers(0, 200))
        rep = int(rng.integers(0, K))
        assert pkg.layup_peer(seed, step, layer, rep, K) == oracle.peer(seed, step, layer, rep, K, 0)
        assert pkg.layup_peer(seed, step, -1, rep, K) == oracle.peer(seed, step, layer, rep, K, 1)
    with pytest.raises(pkg.LayUpError):
        pkg.layup_peer(0, 0, 0, 0, 1)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_means_loud_failure_not_fallback(lib):
    with pytest.raises(pkg.LayUpError) as e:
        pkg.LayUp(4, [100], 0.01)
    assert e.value.code == pkg.LAYUP_ECUDA
    # and straight through the C-ABI: init must report a CUDA error, never succeed
    arr = (ctypes.c_int64 * 1)(100)
    cfg = binding._Config(4, 1, arr, 0.01, 0.0, 0, 0, 0.0, 0)
    ctx = ctypes.c_void_p()
    rc = lib.layup_init(ctypes.byref(cfg), ctypes.c_void_p(128), 1 << 20, ctypes.byref(ctx))
    assert rc == pkg.LAYUP_ECUDA and not ctx.value
    assert b"cuda" in lib.layup_last_error(None).lower()


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2410_05985_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "layup_oracle" not in src and "curand" not in src.lower().replace("does not include curand", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2410_05985_b200\b", src, flags=re.M), f
            assert "#include \"../paper" not in src


def test_header_is_plain_c(tmp_path):
    """include/layup.h is a C boundary: it compiles as C99 with no C++ or torch types in it."""
    import subprocess
    src = tmp_path / "use_layup.c"
    src.write_text('#include "layup.h"\n'
                   'int probe(void) { layup_config c; size_t n = 0; c.K = 1; c.L = 0; c.numel = 0;\n'
                   '  return layup_arena_bytes(&c, &n) == LAYUP_EINVAL ? (int)sizeof(c) : -1; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                           "-c", str(src), "-o", str(tmp_path / "use_layup.o")])


def _cc(tmp_path, defines, libs):
    exe = str(tmp_path / ("c_abi" + ("_layout" if defines else "")))
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    csrc = os.path.join(ROOT, "paper_2410_05985_b200", "csrc")
    cmd = ["gcc", "-std=gnu99", "-Wall", "-Werror", "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(cuda, "include")] + \
          defines + [os.path.join(ROOT, "tests", "c_abi_driver.c"), "-o", exe]
    if libs:
        cmd += ["-L" + csrc, "-llayup", "-L" + os.path.join(cuda, "lib64"), "-lcudart",
                "-Wl,-rpath," + csrc, "-Wl,-rpath," + os.path.join(cuda, "lib64")]
    import subprocess
    subprocess.check_call(cmd)
    return exe


def test_struct_layout_seen_by_a_c_compiler_matches_the_ctypes_mirror(tmp_path):
    """sizeof / offsetof of layup_config and layup_tuning as gcc lays them out (tests/c_abi_driver.c
    -DLAYOUT_ONLY) against binding._Config / _Tuning: the Python mirror is hand-written."""
    import subprocess
    out = subprocess.run([_cc(tmp_path, ["-DLAYOUT_ONLY"], False)], capture_output=True, text=True, check=True).stdout
    got = dict(line.split() for line in out.splitlines())
    assert int(got.pop("sizeof.layup_config")) == ctypes.sizeof(binding._Config)
    assert int(got.pop("sizeof.layup_tuning")) == ctypes.sizeof(binding._Tuning)
    want = {"layup_config.%s" % n: getattr(binding._Config, n).offset for n, _ in binding._Config._fields_}
    want.update({"layup_tuning.%s" % n: getattr(binding._Tuning, n).offset for n, _ in binding._Tuning._fields_})
    assert {k: int(v) for k, v in got.items()} == want


def test_c_program_links_against_the_library(lib, tmp_path):
    """The compute half of tests/c_abi_driver.c builds and links against liblayup.so here; it RUNS in
    tests/test_zy_c_abi_gpu.py on the GPU box.  Without a device it must fail loudly, not fall back."""
    import subprocess
    exe = _cc(tmp_path, [], True)
    if not torch.cuda.is_available():
        r = subprocess.run([exe], capture_output=True, text=True)
        assert r.returncode != 0 and "C_ABI_OK" not in r.stdout
