"""CPU-only: the C-ABI library builds, loads and exports every symbol include/dyplan.h declares; the ctypes
mirrors of its structs match the header; no compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "include", "dyplan.h")


@pytest.fixture(scope="module")
def binding():
    from paper_2607_02942_b200 import build
    build.build()
    from paper_2607_02942_b200 import binding as b
    return b


def declared():
    src = open(HDR).read()
    return sorted(set(re.findall(r"^DYPLAN_API\s+[\w\s\*]+?\b(dyplan_\w+)\s*\(", src, flags=re.M)))


def test_header_declares_the_three_calls():
    names = declared()
    for n in ("dyplan_compile", "dyplan_replan", "dyplan_select", "dyplan_create", "dyplan_destroy"):
        assert n in names
    assert "dyplan_switch" in names
    assert "dyplan_compile_linear" in names
    assert "dyplan_bind" in names
    assert "dyplan_set_flags" in names
    assert "dyplan_measure_issue_rates" in names
    assert "dyplan_compile_static" in names
    assert len(names) == 19


def test_library_exports_every_declared_symbol(binding):
    l = binding.lib()
    for n in declared():
        assert hasattr(l, n), n
    assert sorted(binding.EXPORTS) == declared()
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r" T (dyplan_\w+)", out)))
    assert exported == declared()          # nothing else leaks out of the library


def test_struct_mirrors_match_header(binding):
    # compile a tiny C program against the header and compare sizeof / offsetof with the ctypes mirrors
    import tempfile
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "dyplan.h"
int main(void) {
  printf("%zu %zu %zu\n", sizeof(dyplan_batch), sizeof(dyplan_bundle), sizeof(dyplan_stats));
  printf("%zu %zu %zu %zu\n", offsetof(dyplan_batch, node_off), offsetof(dyplan_batch, cap), offsetof(dyplan_bundle, corr64), offsetof(dyplan_stats, score_ms));
  return 0;
}'''
    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "t.c")
        open(src, "w").write(prog)
        exe = os.path.join(d, "t")
        subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", exe, src])
        a, b = subprocess.check_output([exe], text=True).strip().split("\n")
    sizes = [int(x) for x in a.split()]
    offs = [int(x) for x in b.split()]
    assert sizes == [C.sizeof(binding.CBatch), C.sizeof(binding.CBundle), C.sizeof(binding.CStats)]
    assert offs == [binding.CBatch.node_off.offset, binding.CBatch.cap.offset, binding.CBundle.corr64.offset,
                    binding.CStats.score_ms.offset]


def test_strerror_and_version_without_a_device(binding):
    assert binding.dyplan_version() >= 100
    assert binding.dyplan_strerror(0) == "ok"
    assert "NULL" in binding.dyplan_strerror(binding.ERR_NULL)


def test_create_fails_loudly_without_a_device(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(binding.DyplanError) as e:
        binding.Context(0)
    assert e.value.code == binding.ERR_CUDA       # no CPU fallback


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_02942_b200")
    for dp, _dn, fns in os.walk(pkg):
        if "build" in dp.split(os.sep)[-1:]:
            continue
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "dyplan_oracle" not in src and "liborc" not in src, fn
