"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a without a GPU, loads,
and exports every symbol include/uep.h declares.  No compute call is made here."""
import ctypes
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "uep.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(uep_[a-z_]+)\s*\(", src)))


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "uep.h"\nint main(void){uep_config c; (void)c; return UEP_OK;}\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-fsyntax-only",
                           "-I", os.path.join(ROOT, "include"), str(c)])


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2606_04101_b200 import build, binding
    path = build.build()
    L = ctypes.CDLL(path)
    names = _declared()
    assert {"uep_histogram", "uep_plan", "uep_remap", "uep_pack", "uep_balance", "uep_create",
            "uep_destroy", "uep_workspace_bytes", "uep_plan_bytes", "uep_strerror"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"{n} declared in uep.h but not exported"
    assert sorted(binding.EXPORTS) == names
    L.uep_strerror.restype = ctypes.c_char_p
    assert L.uep_strerror(0) == b"ok" and b"invalid" in L.uep_strerror(-1)


def test_built_for_sm_100a_only():
    from paper_2606_04101_b200 import build
    out = subprocess.check_output(["cuobjdump", "-lelf", build.build()], text=True)
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    from paper_2606_04101_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "missing.so"))
    try:
        binding.lib()
    except binding.UepError as e:
        assert "no CPU fallback" in str(e)
    else:
        raise AssertionError("binding.lib() must raise when libuep.so is missing")


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_04101_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "uep_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_04101_b200\b", txt, flags=re.M)
            assert '#include "uep' not in txt.replace('#include "uep_oracle', "")
