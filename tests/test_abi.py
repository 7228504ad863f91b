"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/symdel.h declares; host-only entry points behave; the product never imports the oracle."""
import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2403_09010_b200 import build, symdel

    build.build_native()
    return symdel.lib()


def declared_symbols():
    text = (ROOT / "include" / "symdel.h").read_text()
    return sorted(set(re.findall(r"SYMDEL_API\s+[\w\s\*]+?\b(symdel_\w+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = declared_symbols()
    for must in ("symdel_self", "symdel_cross", "symdel_self_host", "symdel_cross_host", "symdel_workspace_bytes",
                 "symdel_create", "symdel_destroy", "symdel_strerror", "symdel_get_stats"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2403_09010_b200 import symdel

    names = declared_symbols()
    assert sorted(symdel.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", str(ROOT / "paper_2403_09010_b200" / "libsymdel.so")],
                         capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (symdel_\w+)", out))
    assert exported == set(names)  # nothing else leaks, nothing is missing


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "symdel.h"\nint main(void){ symdel_stats s; (void)s; return SYMDEL_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", str(ROOT / "include"), "-c", str(src), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_strerror_and_workspace_arithmetic(lib):
    from paper_2403_09010_b200 import symdel

    assert lib.symdel_strerror(0) == b"ok"
    for code in range(-9, 0):
        assert lib.symdel_strerror(code) not in (b"", b"unknown error")
    a = symdel.symdel_workspace_bytes(1000, 15000, 0, 0, 24, 2, 0)
    b = symdel.symdel_workspace_bytes(2000, 30000, 0, 0, 24, 2, 0)
    c = symdel.symdel_workspace_bytes(1000, 15000, 0, 0, 24, 3, 0)
    assert 0 < a < b and a < c
    with pytest.raises(symdel.SymdelError):
        symdel.symdel_workspace_bytes(10, 100, 0, 0, 24, 9)  # d > D_MAX
    with pytest.raises(symdel.SymdelError):
        symdel.symdel_workspace_bytes(10, 100, 0, 0, 65, 2)  # max_len > L_MAX


def test_stats_struct_matches_header(lib):
    from paper_2403_09010_b200 import symdel

    text = (ROOT / "include" / "symdel.h").read_text()
    body = text[text.index("typedef struct {"):text.index("} symdel_stats;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split("{", 1)[1].split(";"):
        decl = decl.strip()
        if decl:
            names = decl.split(None, 1)[1]
            fields += [n.strip() for n in names.split(",")]
    assert fields == [f for f, _ in symdel.Stats._fields_]


def test_no_gpu_fails_loudly(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2403_09010_b200 import symdel

    with pytest.raises(symdel.SymdelError):
        symdel.Context(0)  # SYMDEL_E_CUDA: no device, and no CPU fallback


def test_product_never_touches_the_oracle():
    """Neither side imports, includes or loads the other (shared: only the input generator)."""
    import re

    bad = (re.compile(r"^\s*(import|from)\s"), re.compile(r"#\s*include"), re.compile(r"CDLL|dlopen|LoadLibrary"))
    hit = lambda ln: any(b.search(ln) for b in bad)
    for p in list((ROOT / "paper_2403_09010_b200").rglob("*.py")) + list((ROOT / "paper_2403_09010_b200" / "csrc").glob("*")):
        for ln in p.read_text(errors="ignore").splitlines():
            assert not ("oracle" in ln and hit(ln)), (p, ln)
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".cpp"):
            for ln in p.read_text().splitlines():
                assert not (("symdel" in ln or "paper_2403_09010_b200" in ln or "csrc" in ln) and hit(ln)), (p, ln)


def test_no_process_global_init_state_in_the_library():
    """Constant tables and kernel attributes belong to a device: they are set up by symdel_create for the
    context's device (include/symdel.h "Devices and threads"), never behind a process-wide flag, and no tuning
    knob lives in a global variable.  Source check (the two-context run is in the GPU tests)."""
    csrc = ROOT / "paper_2403_09010_b200" / "csrc"
    for p in sorted(csrc.glob("*")):
        text = re.sub(r"//.*", "", p.read_text())
        assert not re.search(r"\bstatic\s+(bool|int|u32|cudaError_t)\s+\w+\s*(=|;)", text), p  # no static flags
        assert not re.search(r"^\s*(int|bool|u32)\s+g_\w+", text, flags=re.M), p               # no global knobs
    api = (csrc / "symdel_api.cu").read_text()
    create = api[api.index("int symdel_create("):api.index("void symdel_destroy(")]
    for setup in ("sd_generate_setup", "sd_sort_setup", "sd_join_setup"):
        assert setup in create, setup
    build_py = (ROOT / "paper_2403_09010_b200" / "build.py").read_text()
    assert "environ" not in build_py  # build() compiles exactly what is committed: no environment hook


def test_kernel_sources_carry_no_tuning_bench():
    """The swept tunables are frozen: no #ifndef-overridable macro, debug path or variant sweep in csrc/."""
    csrc = ROOT / "paper_2403_09010_b200" / "csrc"
    for p in sorted(csrc.glob("*")):
        text = p.read_text()
        assert "#ifndef" not in text and "OS_DBG" not in text and "OS_SWEEP" not in text, p
