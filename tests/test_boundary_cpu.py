"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/xy.h declares; host-only argument logic works without a GPU; product code never touches
the oracle."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1210_6116_b200 import build
    return C.CDLL(build.build())


def declared_functions():
    text = open(os.path.join(ROOT, "include", "xy.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(xy_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_five_calls():
    names = declared_functions()
    for n in ("xy_create", "xy_sw_sweeps", "xy_measure", "xy_pcc_run", "xy_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n


def test_binding_covers_every_declared_symbol(lib):
    from paper_1210_6116_b200 import binding
    assert sorted(binding.EXPORTED) == declared_functions()


def test_workspace_bytes_and_argument_errors(lib):
    n = C.c_size_t()
    lib.xy_last_error.restype = C.c_char_p
    assert lib.xy_workspace_bytes(64, 0, C.byref(n)) == 0
    small = n.value
    assert small >= 64 * 64 * (4 + 4) + 64 * 64 // 4
    assert lib.xy_workspace_bytes(65536, 0, C.byref(n)) == 0
    assert 32 * 2 ** 30 < n.value < 34 * 2 ** 30            # theta 16 GiB + u32 labels 16 GiB + bonds 1 GiB
    assert lib.xy_workspace_bytes(65536, 1, C.byref(n)) == 0
    assert 48 * 2 ** 30 < n.value < 50 * 2 ** 30            # with 64-bit labels
    for bad in (0, 1, 63, 96, 65536 + 64):
        assert lib.xy_workspace_bytes(bad, 0, C.byref(n)) == -2
        assert b"unsupported" in lib.xy_last_error()
    assert lib.xy_workspace_bytes(64, 99, C.byref(n)) == -1
    assert lib.xy_workspace_bytes(64, 0, None) == -1


def test_xi2nd_is_eq8(lib):
    """xy_xi2nd (host arithmetic, no GPU): Eq. 8 against closed forms -- an Ornstein-Zernike propagator
    chi(k) = A / (xi^-2 + 4 sin^2(k/2)) returns its own xi exactly -- and against Table I's row L = 64 through the
    oracle-free inversion chi0 / chik = 1 + (2 sin(pi/L) xi)^2"""
    import math
    lib.xy_xi2nd.argtypes = [C.c_double, C.c_double, C.c_uint32, C.POINTER(C.c_double)]
    out = C.c_double()
    for L in (64, 4096, 65536):
        for xi in (0.3 * L, 0.7506912 * L, 5.0):
            khat2 = 4.0 * math.sin(math.pi / L) ** 2
            chi0, chik = 1.0 / xi ** -2, 1.0 / (xi ** -2 + khat2)
            assert lib.xy_xi2nd(chi0, chik, L, C.byref(out)) == 0
            assert out.value == pytest.approx(xi, rel=1e-9)
    assert lib.xy_xi2nd(1.0, 0.0, 64, C.byref(out)) == -1 and math.isnan(out.value)
    assert lib.xy_xi2nd(1.0, 2.0, 64, C.byref(out)) == -1
    assert lib.xy_xi2nd(float("nan"), 1.0, 64, C.byref(out)) == -1
    assert lib.xy_xi2nd(2.0, 1.0, 1, C.byref(out)) == -1
    assert lib.xy_xi2nd(2.0, 1.0, 64, None) == -1


def test_no_cpu_fallback(lib):
    """without a CUDA device xy_create must fail loudly, never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    lib.xy_create.argtypes = [C.POINTER(C.c_void_p), C.c_uint32, C.c_uint64, C.c_int]
    assert lib.xy_create(C.byref(h), 64, 1, 0) == -4
    assert not h.value
    import paper_1210_6116_b200 as m
    with pytest.raises(m.XYError):
        m.XYState(64, 1)


def test_product_code_is_independent_of_the_oracle():
    pkg = os.path.join(ROOT, "paper_1210_6116_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "xy_oracle" not in src and "xyo_" not in src, f
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    osrc = open(os.path.join(ROOT, "oracle", "xy_oracle.c")).read()
    assert "cuda" not in re.sub(r"/\*.*?\*/", "", osrc, flags=re.S).lower()
    assert "#include \"" not in osrc                      # no project headers shared with the CUDA path


def test_struct_layouts_match_the_header(tmp_path):
    """sizeof / offsetof of every struct of include/xy.h as a C compiler sees them against the ctypes mirrors of the
    binding (a silent mismatch would corrupt records without failing a call)."""
    import subprocess
    from paper_1210_6116_b200 import binding as b
    pairs = {"xy_obs": b.Obs, "xy_fourier": b.Fourier, "xy_pcc_schedule": b.PccSchedule, "xy_pcc_out": b._PccOut,
             "xy_pcc_state": b.PccState, "xy_potts_obs": b.PottsObs}
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{os.path.join(ROOT, "include", "xy.h")}"', 'int main(void) {']
    for cname, cls in pairs.items():
        lines.append(f'printf("{cname} %zu", sizeof({cname}));')
        for fname, _ in cls._fields_:
            lines.append(f'printf(" %zu", offsetof({cname}, {fname}));')
        lines.append('printf("\\n");')
    lines += ['return 0; }']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.strip().splitlines()
    assert len(out) == len(pairs)
    for line in out:
        name, size, *offs = line.split()
        cls = pairs[name]
        assert int(size) == C.sizeof(cls), name
        assert [int(o) for o in offs] == [getattr(cls, f).offset for f, _ in cls._fields_], name
