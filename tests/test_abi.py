"""Boundary checks that need no GPU: the C-ABI library builds for sm_100a, loads, exports exactly the
symbols include/soma.h declares, the Python mirror of `soma_params` has the C layout, parameter
validation works, and the product path fails loudly (no CPU fallback) when no device is there."""
import ctypes as C
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]
HEADER = ROOT / "include" / "soma.h"


@pytest.fixture(scope="module")
def soma():
    import __graft_entry__ as entry
    entry.build()
    import paper_2606_09356_b200 as soma
    soma.load_library()
    return soma


def _declared_functions():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(soma_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(soma):
    declared = _declared_functions()
    assert len(declared) >= 6
    for must in ("soma_create", "soma_load_state", "soma_mc_steps", "soma_get_density", "soma_get_positions", "soma_destroy"):
        assert must in declared                     # the six names north_star lists
    nm = subprocess.run(["nm", "-D", "--defined-only", str(soma.LIB_PATH)], capture_output=True, text=True, check=True).stdout
    exported = sorted(set(re.findall(r"\bT (soma_[a-z_0-9]+)\b", nm)))
    assert exported == declared
    assert sorted(soma.EXPORTS) == declared
    lib = soma.load_library()
    for name in declared:
        assert hasattr(lib, name)


def test_library_holds_sm_100a_code_only(soma):
    out = subprocess.run(["cuobjdump", "-lelf", str(soma.LIB_PATH)], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_params_struct_layout_matches_the_header(soma, tmp_path):
    fields = [f[0] for f in soma.soma_params._fields_]
    src = tmp_path / "layout.c"
    body = "\n".join(f'  printf("{f} %zu\\n", offsetof(soma_params, {f}));' for f in fields)
    src.write_text(f'#include <stdio.h>\n#include <stddef.h>\n#include "{HEADER}"\nint main(void) {{\n{body}\n'
                   '  printf("sizeof %zu\\n", sizeof(soma_params));\n  return 0;\n}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", str(src), "-o", str(exe)], check=True)   # header is plain C
    got = dict(line.split() for line in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for f in fields:
        assert int(got[f]) == getattr(soma.soma_params, f).offset, f
    assert int(got["sizeof"]) == C.sizeof(soma.soma_params)


def _params(soma, **over):
    kw = dict(n_chains=256, beads_per_chain=32, n_types=2, type_patterns=np.array([[0] * 16 + [1] * 16], dtype=np.uint8),
              chain_pattern=None, b=1.0, chiN=np.array([[0, 20], [20, 0]], dtype=np.float32), kappaN=50.0,
              grid=(16, 16, 16), box=(8.0, 8.0, 8.0), move_halfwidth=0.5, seed=1)
    kw.update(over)
    return soma.make_params(**kw)


def test_workspace_bytes_and_validation(soma):
    p, keep = _params(soma)
    nbytes = soma.soma_workspace_bytes(p)
    B, TC = 256 * 32, 2 * 16 ** 3
    assert nbytes >= 2 * 3 * 4 * B + 3 * 4 * TC + 5 * 256          # two position sets, two count grids, omega, tables
    assert nbytes < 2 * (2 * 3 * 4 * B + 4 * 4 * TC) + 40 * 256   # + external field, sort scratch, alignment
    bad = [
        dict(n_chains=0), dict(beads_per_chain=0), dict(n_types=9), dict(b=0.0), dict(grid=(16, 0, 16)),
        dict(box=(8.0, -1.0, 8.0)), dict(chiN=np.array([[0, 20], [19, 0]], dtype=np.float32)),
        dict(chiN=np.array([[1, 20], [20, 0]], dtype=np.float32)),
        dict(type_patterns=np.array([[0] * 16 + [2] * 16], dtype=np.uint8)),
        dict(chain_pattern=np.full(256, 1, dtype=np.uint8)), dict(move_halfwidth=float("nan")),
    ]
    for over in bad:
        q, keep2 = _params(soma, **over)
        assert soma.soma_workspace_bytes(q) == 0, over
        assert soma.load_library().soma_last_error(None) != b""


def test_null_handle_calls_are_rejected_not_crashing(soma):
    lib = soma.load_library()
    assert lib.soma_destroy(None) == soma.SOMA_OK
    assert lib.soma_mc_steps(None, 1, None) == soma.SOMA_EINVAL
    assert lib.soma_get_density(None, None, 0) == soma.SOMA_EINVAL
    assert lib.soma_get_positions(None, None, None, None, 0) == soma.SOMA_EINVAL
    assert lib.soma_load_state(None, None, None, None, 0, 0) == soma.SOMA_EINVAL
    out = C.c_void_p(123)
    assert lib.soma_create(None, None, C.byref(out)) == soma.SOMA_EINVAL and out.value is None


def test_no_cpu_fallback_without_a_device(soma):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present; the fail-loudly path is for boxes without one")
    p, keep = _params(soma)
    with pytest.raises(soma.SomaError) as e:
        soma.soma_create(p, 0)
    assert e.value.code == soma.SOMA_ECUDA
    with pytest.raises(soma.SomaError):
        soma.Soma(256, 32, 2, keep[0], None, 1.0, keep[2], 50.0, (16, 16, 16), (8.0,) * 3, 0.5, 1)


def test_product_package_never_touches_the_oracle():
    # The product path may not import, call or link anything under oracle/ (and vice versa).
    pkg = ROOT / "paper_2606_09356_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [HEADER]:
        text = f.read_text()
        assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
        assert not re.search(r"#\s*include[^\n]*oracle", text), f
        assert "libscmf_oracle" not in text and "scmf_oracle.cpp" not in text, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".cpp", ".h"):
            text = f.read_text()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_09356_b200\b", text, flags=re.M), f
            assert not re.search(r"#\s*include[^\n]*(soma|paper_2606)", text), f
            assert "libsoma_b200" not in text, f


def test_noalloc_entry_point_refuses_oversized_and_malformed_calls_before_touching_a_device(soma):
    """soma_validate_noalloc checks its sizes against the fixed scratch array before any CUDA call, so the refusal -- and
    its message, which has to tell a caller who cannot allocate what the limit is -- can be checked without a GPU.  The
    pointers are never dereferenced on this path."""
    lib = soma.load_library()
    dummy = np.zeros(8, dtype=np.float32)
    ptr = dummy.ctypes.data
    v = soma.soma_validation()
    err = C.create_string_buffer(512)

    def call(n_chains, N, counts=None, T=0, cells=0, x=ptr, out=C.byref(v)):
        return lib.soma_validate_noalloc(x, ptr, ptr, n_chains, N, counts, T, cells, None, out, err, len(err))

    assert call((1 << 28) // 32 + 1, 32) == soma.SOMA_EINVAL            # one chain more than 2^28 beads
    assert b"268435456" in err.value and b"scratch" in err.value
    assert call(1 << 40, 65535) == soma.SOMA_EINVAL                      # no overflow in the size check
    assert call(0, 32) == soma.SOMA_EINVAL and call(4, 0) == soma.SOMA_EINVAL
    assert call(4, 2, x=None) == soma.SOMA_EINVAL and call(4, 2, out=None) == soma.SOMA_EINVAL
    assert call(4, 2, counts=ptr, T=9, cells=8) == soma.SOMA_EINVAL      # the report has eight per-type fields
    assert call(4, 2, counts=ptr, T=2, cells=1 << 31) == soma.SOMA_EINVAL
    assert lib.soma_validate_noalloc(ptr, ptr, ptr, 1 << 30, 32, None, 0, 0, None, C.byref(v), None, 0) == soma.SOMA_EINVAL   # errbuf is optional
