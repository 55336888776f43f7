"""`-m "not gpu"`: the C-ABI library loads and exports every symbol include/gpuann.h declares, the ctypes structure
matches the header, and (without a GPU) the entry points fail loudly instead of falling back to a CPU path."""
import ctypes as C
import re
from pathlib import Path

import pytest

from paper_2402_18858_b200 import binding as B
from paper_2402_18858_b200 import build as BUILD

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "gpuann.h").read_text()


@pytest.fixture(scope="module")
def lib():
    BUILD.build()
    return B.lib()


def declared_symbols():
    code = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    return sorted(set(re.findall(r"\b(gpuann_[a-z0-9_]+)\s*\(", code)))


def test_header_and_binding_list_the_same_symbols():
    assert declared_symbols() == sorted(B.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"libgpuann.so does not export {name}"


def test_params_struct_matches_header():
    code = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    body = re.search(r"typedef struct \{(.*?)\} gpuann_params;", code, flags=re.S).group(1)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        typ, names = decl.rsplit(" ", 1)[0], decl.split(" ", 1)[1]
        for nm in names.split(","):
            fields.append((nm.strip().split()[-1], typ.split()[0]))
    ctypes_of = {"int": C.c_int, "double": C.c_double, "int64_t": C.c_int64}
    assert [(n, ctypes_of[t]) for n, t in fields] == [(n, t) for n, t in B.gpuann_params._fields_]


def test_default_params(lib):
    p = B.gpuann_default_params()
    assert (p.precision, p.newton_max_iter, p.newton_tol, p.T_min, p.T_max, p.T_active, p.device, p.chunk_cells) == \
        (B.GPUANN_PRECISION_BF16, 20, 1e-6, 200.0, 3500.0, 0.0, -1, 0)


def test_timing_class_names(lib):
    n = lib.gpuann_timing_num_classes()
    names = [lib.gpuann_timing_class_name(i).decode() for i in range(n)]
    assert len(set(names)) == n and all(names)
    assert lib.gpuann_timing_class_name(n) == b""


def test_no_cpu_fallback_and_null_checks(lib):
    import torch
    out = C.c_void_p(0)
    assert lib.gpuann_create(None, None) == B.GPUANN_ERR_INVALID_ARG
    assert b"out is NULL" in lib.gpuann_last_error(None)
    if not torch.cuda.is_available():
        st = lib.gpuann_create(None, C.byref(out))
        assert st == B.GPUANN_ERR_UNSUPPORTED and not out.value
        assert b"no CPU fallback" in lib.gpuann_last_error(None)
        with pytest.raises(B.GpuannError):
            B.gpuann_create()
    assert lib.gpuann_chem_step(None, 0, None, None, None, None, 1e-6, None) == B.GPUANN_ERR_INVALID_ARG
    assert lib.gpuann_input_moments_static(None, 1, 1, None, None, None, 0.1, None, None, None) == B.GPUANN_ERR_INVALID_ARG
    assert lib.gpuann_destroy(None) == B.GPUANN_OK
    assert lib.gpuann_launch_count(None) == 0


def test_static_scratch_limits_match_the_header():
    """GPUANN_STATIC_MAX_SPECIES / GPUANN_STATIC_SCRATCH_BYTES: header, binding and the layout the header states
    ((512 blocks x (64 + 2) features + 2 x 66) doubles) agree; k_aux.cu static_asserts the same two numbers."""
    hdr = {m.group(1): int(m.group(2)) for m in re.finditer(r"#define (GPUANN_STATIC_\w+) (\d+)", HEADER)}
    assert hdr == {"GPUANN_STATIC_MAX_SPECIES": B.GPUANN_STATIC_MAX_SPECIES, "GPUANN_STATIC_SCRATCH_BYTES": B.GPUANN_STATIC_SCRATCH_BYTES}
    d = B.GPUANN_STATIC_MAX_SPECIES + 2
    assert B.GPUANN_STATIC_SCRATCH_BYTES == (512 * d + 2 * d) * 8


def test_debug_library_has_the_same_abi():
    """libgpuann_debug.so (build.py --debug: -DGPUANN_DEBUG_SPIN) exports every symbol the header declares; skipped when
    it has not been built (__graft_entry__.build() builds it)."""
    if not BUILD.LIB_DEBUG.exists() or BUILD.needs_build(BUILD.LIB_DEBUG):
        pytest.skip("libgpuann_debug.so not built or out of date")
    dbg = C.CDLL(str(BUILD.LIB_DEBUG))
    for name in declared_symbols():
        assert hasattr(dbg, name), f"libgpuann_debug.so does not export {name}"
