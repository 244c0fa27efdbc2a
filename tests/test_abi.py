"""The C-ABI shared library builds for sm_100a without a GPU, loads, and exports every entry
point include/cfgms.h declares (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "cfgms.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cfgms_[a-z_]+)\s*\(", src)))


def test_library_builds_and_exports_header_symbols():
    from paper_2607_02119_b200.build import build_lib
    import paper_2607_02119_b200 as pkg
    path = build_lib()
    lib = C.CDLL(path)
    names = _declared()
    assert {"cfgms_create", "cfgms_step", "cfgms_deinterleave"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in cfgms.h but not exported"
    assert set(pkg.EXPORTS) == set(names)


def test_measurement_probes_are_not_part_of_the_abi():
    """The design-choice probes (one of which produces wrong tokens by design) live in a separate build of the
    library (-DCFGMS_PROBES), not in the public header, the binding's constants or the product library's strings."""
    import paper_2607_02119_b200 as pkg
    from paper_2607_02119_b200 import binding
    header = open(os.path.join(ROOT, "include", "cfgms.h")).read()
    assert "PROBE" not in header
    assert not [n for n in dir(binding) if "PROBE" in n]
    assert "probes" not in pkg.version()


def test_version_and_strerror_strings():
    import paper_2607_02119_b200 as pkg
    assert "sm_100a" in pkg.version()
    lib = pkg.library()
    assert lib.cfgms_strerror(0) == b"ok"
    assert b"fallback" in lib.cfgms_strerror(5)


def test_struct_layouts_match_header(tmp_path):
    # the C compiler's view of include/cfgms.h (LP64) against the ctypes mirrors, field by field
    import os
    import subprocess
    from paper_2607_02119_b200 import binding as b
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    structs = {"cfgms_config": b.cfgms_config, "cfgms_step_args": b.cfgms_step_args, "cfgms_info": b.cfgms_info}
    lines = []
    for name, cls in structs.items():
        lines.append(f'printf("{name} %zu\\n", sizeof({name}));')
        for field, _ in cls._fields_:
            lines.append(f'printf("{name}.{field} %zu\\n", offsetof({name}, {field}));')
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "cfgms.h"\nint main(void) {\n' + "\n".join(lines) + "\nreturn 0; }\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(root, "include"), "-o", str(exe), str(src)], check=True)
    out = dict(l.split() for l in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    for name, cls in structs.items():
        assert int(out[name]) == C.sizeof(cls), name
        for field, _ in cls._fields_:
            assert int(out[f"{name}.{field}"]) == getattr(cls, field).offset, f"{name}.{field}"
    assert b.cfgms_step_args.seed.offset == 48 and b.cfgms_step_args.hidden.offset == 0


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2607_02119_b200 as pkg
    h = torch.zeros(1, 8, 8, dtype=torch.bfloat16)
    with pytest.raises((ValueError, pkg.CfgmsError)):
        pkg.Context(h, torch.zeros(1, 8, dtype=torch.bfloat16))
    # straight through the ABI: a non-null pointer on a machine without a device is an error, not a fallback
    out = C.c_void_p()
    rc = pkg.library().cfgms_create(C.byref(out), 16, 16, 1, 8, 8, None)
    assert rc != 0 and not out.value
