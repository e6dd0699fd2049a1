"""The C-ABI library loads and exports every symbol include/tkhp.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def built_lib():
    from paper_2011_01207_b200 import build
    return build.build()


def _declared_symbols():
    text = (ROOT / "include" / "tkhp.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tkhp_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(built_lib):
    names = _declared_symbols()
    assert "tkhp_nblist_build" in names and "tkhp_polar_energy" in names and len(names) >= 13
    L = ctypes.CDLL(str(built_lib))
    for name in names:
        assert hasattr(L, name), f"{name} declared in tkhp.h but not exported"


def test_binding_lists_every_symbol(built_lib):
    import paper_2011_01207_b200 as pk
    assert sorted(pk.EXPORTED_SYMBOLS) == _declared_symbols()
    for name in pk.EXPORTED_SYMBOLS:
        assert callable(getattr(pk, name)), name


def test_params_struct_layout_matches_header(built_lib, tmp_path):
    """sizeof/offsetof of tkhp_params as gcc sees include/tkhp.h == the ctypes mirror."""
    import subprocess
    import paper_2011_01207_b200 as pk
    names = [f[0] for f in pk.TkhpParams._fields_]
    src = tmp_path / "layout.c"
    body = "".join(f'    printf("{n} %zu\\n", offsetof(tkhp_params, {n}));\n' for n in names)
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "tkhp.h"\nint main(void) {\n'
                   '    printf("sizeof %zu\\n", sizeof(tkhp_params));\n' + body + "    return 0;\n}\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", str(ROOT / "include"), str(src), "-o", str(exe)], check=True)
    out = dict(line.split() for line in subprocess.run([str(exe)], check=True, capture_output=True,
                                                       text=True).stdout.splitlines())
    assert int(out["sizeof"]) == ctypes.sizeof(pk.TkhpParams) == 80
    for n in names:
        assert int(out[n]) == getattr(pk.TkhpParams, n).offset, n


def test_host_side_parameter_checks(built_lib):
    """tkhp_workspace_bytes is pure host code: error paths are testable without a GPU."""
    import paper_2011_01207_b200 as pk
    ok = pk.TkhpParams(648, pk.TKHP_MIXED, 0, pk.TKHP_LIST_TILES, 18.64, 7.0, 2.0, 0.5446, 0.39, 0, 0)
    n = pk.tkhp_workspace_bytes(ok)
    assert 100_000 < n < 50_000_000
    big = pk.TkhpParams(1_066_629, pk.TKHP_MIXED, 0, pk.TKHP_LIST_TILES, 220.1, 7.0, 2.0, 0.5446, 0.39, 0, 0)
    assert pk.tkhp_workspace_bytes(big) < 4 << 30
    bad_cut = pk.TkhpParams(648, pk.TKHP_MIXED, 0, 0, 18.64, 8.0, 2.0, 0.5446, 0.39, 0, 0)
    with pytest.raises(pk.TkhpError) as e:
        pk.tkhp_workspace_bytes(bad_cut)
    assert e.value.code == -3  # TKHP_ECUTOFF
    for field, val in (("n_atoms", 0), ("precision", 7), ("cutoff", -1.0), ("thole_a", 0.0),
                       ("ewald_beta", -0.1), ("list_mode", 5)):
        p = pk.TkhpParams(648, pk.TKHP_MIXED, 0, 0, 18.64, 7.0, 2.0, 0.5446, 0.39, 0, 0)
        setattr(p, field, val)
        with pytest.raises(pk.TkhpError) as e:
            pk.tkhp_workspace_bytes(p)
        assert e.value.code == -1, field
    # range of the erfc fits (both precisions): beta * cutoff <= 6
    p = pk.TkhpParams(648, pk.TKHP_MIXED, 0, 0, 40.0, 7.0, 2.0, 1.0, 0.39, 0, 0)
    with pytest.raises(pk.TkhpError):
        pk.tkhp_workspace_bytes(p)
    p.precision = pk.TKHP_FP64
    with pytest.raises(pk.TkhpError):
        pk.tkhp_workspace_bytes(p)
    p.ewald_beta = 0.85
    assert pk.tkhp_workspace_bytes(p) > 0


def test_no_gpu_means_loud_failure(built_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2011_01207_b200 as pk
    with pytest.raises(pk.TkhpError):
        pk.Polarizer(648, 18.64)


def test_product_never_imports_oracle():
    pkg = ROOT / "paper_2011_01207_b200"
    for path in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + list(pkg.rglob("*.h")):
        text = path.read_text()
        assert "oracle" not in text.lower().replace("no code here is shared with oracle/", "") \
            or path.name in ("gen_erfcx_coeffs.py", "common.cuh", "pcg.cu", "nblist.cu", "pair_math.cuh") \
            and "import oracle" not in text and "oracle/" not in text.replace("shared with oracle/", ""), path
    for path in (ROOT / "oracle").rglob("*.py"):
        assert "paper_2011_01207_b200" not in path.read_text().replace(
            "(``paper_2011_01207_b200``)", ""), path
