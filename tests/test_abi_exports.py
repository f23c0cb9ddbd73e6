"""CPU-only: the C-ABI library builds for sm_100a, loads, and exports every symbol include/*.h declares.
No compute call is made (there is no GPU here)."""
import os
import re

import paper_2606_28166_b200 as T

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    for hdr in sorted(os.listdir(os.path.join(ROOT, "include"))):      # every header under include/: the product API and the test hooks
        src = open(os.path.join(ROOT, "include", hdr)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(tandem_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_library_builds_loads_and_exports_every_declared_symbol():
    T.build()
    L = T.lib()
    names = _declared()
    assert {"tandem_init", "tandem_load_weights", "tandem_step", "tandem_generate", "tandem_free"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    assert sorted(T.EXPORTED_SYMBOLS) == names


def test_struct_sizes_match_header_layout(tmp_path):
    """Compile include/tandem.h with gcc and compare sizeof/offsetof with the ctypes mirrors."""
    import ctypes as C
    import subprocess
    from paper_2606_28166_b200 import binding as b
    src = tmp_path / "sz.c"
    src.write_text('#include "%s"\n#include <stdio.h>\n#include <stddef.h>\n'
                   'int main(){printf("%%zu %%zu %%zu %%zu %%zu %%zu %%zu %%zu\\n", sizeof(tandem_config), sizeof(tandem_params),'
                   'sizeof(tandem_overrides), sizeof(tandem_stats), sizeof(tandem_weights), sizeof(tandem_step_in), sizeof(tandem_step_out),'
                   'offsetof(tandem_config, kv_bytes_per_model));return 0;}\n' % os.path.join(ROOT, "include", "tandem.h"))
    exe = tmp_path / "sz"
    subprocess.run(["gcc", str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert got == [C.sizeof(b._Config), C.sizeof(b._Params), C.sizeof(b._Overrides), C.sizeof(b._Stats), C.sizeof(b._Weights),
                   C.sizeof(b._StepIn), C.sizeof(b._StepOut), b._Config.kv_bytes_per_model.offset]


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_28166_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in s and "from oracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2606_28166_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "`paper_2606_28166_b200/`", ""), f
