"""CPU-side checks of the boundary: libscw.so builds, loads and exports what include/*.h declares."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libscw():
    from paper_2404_07293_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        src = open(h).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(scw_[A-Za-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_header_declares_the_four_named_calls():
    names = declared_symbols()
    for n in ("scw_assemble_spectra", "scw_synthesize_grid", "scw_eval_points", "scw_sweep_wavelengths"):
        assert n in names
    assert len(names) >= 15


def test_library_exports_every_declared_symbol(libscw):
    for n in declared_symbols():
        assert hasattr(libscw, n), f"libscw.so does not export {n}"
    assert libscw.scw_version() >= 100


def test_binding_structs_match_header_layout(libscw, tmp_path):
    """sizeof(scw_layer/scw_modes) as compiled by the C compiler equals the ctypes mirror."""
    import subprocess
    from paper_2404_07293_b200 import binding
    src = tmp_path / "sz.c"
    src.write_text('#include "scwatter.h"\n#include <stdio.h>\n#include <stddef.h>\n'
                   'int main(void){printf("%zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(scw_layer), sizeof(scw_modes),'
                   ' offsetof(scw_layer, gamma), offsetof(scw_modes, p), offsetof(scw_modes, layer),'
                   ' sizeof(scw_exterior), offsetof(scw_exterior, n_re), offsetof(scw_exterior, p_inc));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert int(out[0]) == ctypes.sizeof(binding.scw_layer)
    assert int(out[1]) == ctypes.sizeof(binding.scw_modes)
    assert int(out[2]) == binding.scw_layer.gamma.offset
    assert int(out[3]) == binding.scw_modes.p.offset
    assert int(out[4]) == binding.scw_modes.layer.offset
    assert int(out[5]) == ctypes.sizeof(binding.scw_exterior)
    assert int(out[6]) == binding.scw_exterior.n_re.offset
    assert int(out[7]) == binding.scw_exterior.p_inc.offset
    # the round-2 descriptors
    src2 = tmp_path / "sz2.c"
    src2.write_text('#include "scwatter.h"\n#include <stdio.h>\n#include <stddef.h>\n'
                    'int main(void){printf("%zu %zu %zu %zu %zu %zu %zu\\n", sizeof(scw_window), sizeof(scw_vbuild),'
                    ' offsetof(scw_vbuild, psi), sizeof(scw_stack), offsetof(scw_stack, z_if), offsetof(scw_stack, gamma),'
                    ' offsetof(scw_stack, dir));return 0;}\n')
    exe2 = tmp_path / "sz2"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src2), "-o", str(exe2)], check=True)
    o2 = [int(v) for v in subprocess.run([str(exe2)], capture_output=True, text=True, check=True).stdout.split()]
    assert o2 == [ctypes.sizeof(binding.scw_window), ctypes.sizeof(binding.scw_vbuild), binding.scw_vbuild.psi.offset,
                  ctypes.sizeof(binding.scw_stack), binding.scw_stack.z_if.offset, binding.scw_stack.gamma.offset,
                  binding.scw_stack.dir.offset]
    assert set(binding.EXPORTS) == set(declared_symbols())


def test_null_handles_are_rejected_without_a_gpu(libscw):
    """Entry points that need no device reject NULL contexts (no compute is attempted)."""
    libscw.scw_last_error.restype = ctypes.c_char_p
    assert libscw.scw_destroy(None) == 1
    assert libscw.scw_set_stream(None, None) == 1
    assert libscw.scw_set_workspace(None, None, 0) == 1
    assert libscw.scw_last_error(None) == b"ctx is NULL"
    assert libscw.scw_create(None, 0, None) == 1


def test_product_does_not_import_oracle():
    """The CUDA package and the oracle are independent: neither source tree names the other."""
    pkg = os.path.join(ROOT, "paper_2404_07293_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "scw_oracle" not in txt, f
    for f in glob.glob(os.path.join(ROOT, "oracle", "*")):
        if f.endswith((".py", ".c")):
            txt = open(f).read()
            assert "paper_2404_07293_b200" not in txt.replace("paper_2404_07293_b200/csrc", "") or f.endswith(".c"), f
            assert "import paper_2404_07293_b200" not in txt and "libscw.so" not in txt, f
