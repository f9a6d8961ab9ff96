"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/gpupegas.h declares (no compute calls without a GPU), and it fails loudly, not silently,
when no CUDA device is present."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gpupegas.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gp_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for s in ("gp_create", "gp_set_state", "gp_step", "gp_solve_poisson", "gp_max_dt", "gp_get_state", "gp_destroy"):
        assert s in syms


def test_library_exports_every_declared_symbol():
    from paper_1311_0861_b200 import binding, build
    build.build()
    L = binding.lib()
    for s in declared_symbols():
        assert hasattr(L, s), s
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_1311_0861_b200 as pkg
    with pytest.raises(RuntimeError):
        pkg.Simulation(8, 8, 8, 0.1)
    # and straight through the C ABI
    L = pkg.lib()
    g = pkg.binding.gp_grid(8, 8, 8, 0.1, 1, 0, 1.0)
    b = pkg.binding.gp_bc(0, 0, 0)
    assert not L.gp_create(ctypes.byref(g), 1.4, ctypes.byref(b))
    assert b"no CUDA device" in L.gp_last_error()


def test_product_path_does_not_touch_the_oracle():
    """Nothing under paper_1311_0861_b200/ or bench.py's product arm may import oracle/."""
    pkg_dir = os.path.join(ROOT, "paper_1311_0861_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "liboracle" not in text and "oracle.h" not in text, f


def test_binding_constants_match_the_header():
    """Field ids, component bits and error codes of the ctypes binding are those of include/gpupegas.h."""
    from paper_1311_0861_b200 import binding as B
    text = open(os.path.join(ROOT, "include", "gpupegas.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    values = {}
    for body in re.findall(r"enum\s*\{(.*?)\}", text, flags=re.S):
        nxt = 0
        for item in [x.strip() for x in body.split(",") if x.strip()]:
            name, _, val = [p.strip() for p in item.partition("=")]
            if val:
                nxt = values[val] if val in values else int(val, 0)
            values[name] = nxt
            nxt += 1
    names = ["RHO", "MX", "MY", "MZ", "E", "N", "NUX", "NUY", "NUZ", "EXX", "EXY", "EXZ", "EYY", "EYZ", "EZZ", "PHI",
             "EPS", "PXX", "PXY", "PXZ", "PYY", "PYZ", "PZZ"]
    order = B.FIELDS + B.OD_GAS_FIELDS + B.OD_STAR_FIELDS
    assert len(order) == len(names) == values["GP_NFIELDS_OD"]
    for py_name, c_name in zip(order, names):
        assert B.FIELD_ID[py_name] == values["GP_" + c_name], (py_name, c_name)
    assert (B.GP_GAS, B.GP_STARS, B.GP_OD) == (values["GP_GAS"], values["GP_STARS"], values["GP_OD"])
    define = re.search(r"#define\s+GP_KAPPA_NOALLOC_MAX_CELLS\s+(\d+)", text)
    assert define and int(define.group(1)) == B.KAPPA_NOALLOC_MAX_CELLS == 512 ** 3
    assert (B.GP_ERR_STATE, B.GP_ERR_UNSUPPORTED) == (values["GP_ERR_STATE"], values["GP_ERR_UNSUPPORTED"])
    assert (B.GP_POISSON_PERIODIC, B.GP_POISSON_ISOLATED, B.GP_BC_OUTFLOW) == (
        values["GP_POISSON_PERIODIC"], values["GP_POISSON_ISOLATED"], values["GP_BC_OUTFLOW"])


def test_storage_accounting_is_host_arithmetic():
    """gp_storage_bytes needs no device: state x 2 (ping-pong) + padded Phi + Poisson work arrays; a GP_OD context
    adds two copies of its seven carried fields."""
    import paper_1311_0861_b200 as pkg
    B = pkg.binding
    L = pkg.lib()

    def nbytes(n, comp, poisson):
        g = B.gp_grid(n, n, n, 1.0 / n, comp, poisson, 1.0)
        return L.gp_storage_bytes(ctypes.byref(g))

    n = 64
    cell = 8 * n ** 3
    gas, both = nbytes(n, B.GP_GAS, 0), nbytes(n, B.GP_GAS | B.GP_STARS, 0)
    assert 2 * 5 * cell <= gas <= 2 * 5 * cell + 1.2 * 8 * (n + 34) * (n + 4) ** 2 + (1 << 16)
    assert abs((both - gas) - 2 * 10 * cell) <= 1 << 16
    od = nbytes(n, B.GP_GAS | B.GP_STARS | B.GP_OD, 0)
    assert abs((od - both) - 2 * 7 * cell) <= 1 << 16
    per = nbytes(n, B.GP_GAS | B.GP_STARS, B.GP_POISSON_PERIODIC)
    assert per - both >= 16 * (n // 2 + 1) * n * n + cell          # half spectrum + the source rho + n
    iso = nbytes(n, B.GP_GAS, B.GP_POISSON_ISOLATED)
    assert iso > gas + 4 * cell
    assert L.gp_storage_bytes(None) == 0
