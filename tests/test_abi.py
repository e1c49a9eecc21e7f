"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/osbli.h declares,
its host-only entry points (layout, workspace size, validation, strerror) behave as documented,
and the ctypes structures of the binding match the C structs.  No compute calls (no GPU here)."""
import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "osbli.h"


@pytest.fixture(scope="module")
def osbli():
    from paper_2007_14933_b200 import build
    build.build()
    from paper_2007_14933_b200 import osbli as mod
    return mod


def declared_functions():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(osbli_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(osbli):
    names = declared_functions()
    assert {"osbli_init", "osbli_bc", "osbli_rhs", "osbli_rk3_step"} <= set(names)
    lib = C.CDLL(str(osbli._LIBPATH))
    for name in names:
        assert hasattr(lib, name), f"{name} declared in osbli.h but not exported"
    assert sorted(osbli.EXPORTS) == names


def test_struct_sizes_match_the_c_compiler(osbli, tmp_path):
    src = tmp_path / "sizes.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "osbli.h"\n'
                   'int main(void){printf("%zu %zu %zu %zu %zu %zu\\n", sizeof(osbli_params), sizeof(osbli_metrics),'
                   ' sizeof(osbli_layout), offsetof(osbli_params, bc), offsetof(osbli_params, dirichlet),'
                   ' offsetof(osbli_params, metrics)); return 0;}\n')
    exe = tmp_path / "sizes"
    subprocess.run(["gcc", "-std=c99", "-I", str(ROOT / "include"), str(src), "-o", str(exe)], check=True)
    got = [int(v) for v in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    want = [C.sizeof(osbli.Params), C.sizeof(osbli.Metrics), C.sizeof(osbli.Layout), osbli.Params.bc.offset,
            osbli.Params.dirichlet.offset, osbli.Params.metrics.offset]
    assert got == want


def test_layout_alignment_and_sizes(osbli):
    for n in [(256, 256, 256), (400, 1, 1), (500, 250, 8), (70, 37, 35), (5, 5, 1)]:
        p = osbli.make_params(n=n)
        lay = osbli.osbli_get_layout(p)
        halo = [3 if v > 1 else 0 for v in n]
        assert list(lay.halo) == halo
        assert lay.x_offset % 16 == 0 and lay.stride_y % 16 == 0          # 128-byte aligned rows
        assert lay.stride_y >= lay.x_offset + n[0] + 11                   # halo + the x sweep's tile overhang
        assert lay.stride_z == lay.stride_y * (n[1] + 2 * halo[1])
        assert lay.stride_var == lay.stride_z * (n[2] + 2 * halo[2])
        assert lay.total_doubles == 5 * lay.stride_var
    lay = osbli.osbli_get_layout(osbli.make_params(n=(70, 37, 1), scheme=osbli.SCHEME_WENOZ7))      # 7th order: four ghost points
    assert list(lay.halo) == [4, 4, 0] and lay.stride_y >= lay.x_offset + 70 + 4 and lay.x_offset >= 4
    assert lay.stride_var == lay.stride_y * (37 + 8)
    p = osbli.make_params(n=(512, 512, 512), visc=osbli.VISC_CONST)
    lay = osbli.osbli_get_layout(p)
    assert 5.3e9 < lay.total_doubles * 8 < 6.2e9                          # "about 5.4 GB per state" + halos
    assert osbli.osbli_workspace_bytes(p) == 15 * lay.stride_var * 8      # R + Q2 + Q3 (the fast viscous path stages nothing)
    ex = ((osbli.BC_EXTRAP0,) * 2,) * 3
    assert osbli.osbli_workspace_bytes(osbli.make_params(n=(512, 512, 512), visc=osbli.VISC_CONST, bc=ex)) == 31 * lay.stride_var * 8
    assert osbli.osbli_workspace_bytes(osbli.make_params(n=(512, 512, 512), visc=osbli.VISC_SUTHERLAND, bc=ex)) == 35 * lay.stride_var * 8
    p = osbli.make_params(n=(64, 64, 64), visc=osbli.VISC_SUTHERLAND)
    assert osbli.osbli_workspace_bytes(p) == 35 * osbli.osbli_get_layout(p).stride_var * 8   # + u, v, w, T, mu and their 15 first differences
    p = osbli.make_params(n=(64, 1, 1))
    assert osbli.osbli_workspace_bytes(p) == 15 * osbli.osbli_get_layout(p).stride_var * 8


def test_validation_errors_without_a_gpu(osbli):
    def status(**kw):
        base = dict(n=(16, 16, 16), delta=(0.1, 0.1, 0.1))
        base.update(kw)
        p = osbli.make_params(**base)
        with pytest.raises(osbli.OsbliError) as e:
            osbli.osbli_init(p, 4096, 1 << 40)
        return e.value.status

    assert status(n=(16, 3, 1)) == osbli.EINVAL                            # active direction < 5 points
    assert status(n=(1, 16, 16)) == osbli.EUNSUPPORTED                     # x must be active
    assert status(scheme=7) == osbli.EINVAL
    assert status(gamma=1.0) == osbli.EINVAL
    assert status(eps=1e-30) == osbli.EINVAL
    assert status(bc=((0, 1), (0, 0), (0, 0))) == osbli.EINVAL             # periodic on one side only
    assert status(bc=((2, 1), (0, 0), (0, 0))) == osbli.EINVAL             # Dirichlet without a state
    assert status(bc=((1, 1), (3, 1), (0, 0))) == osbli.EINVAL             # wall without T_w
    assert status(delta=(0.0, 0.1, 0.1)) == osbli.EINVAL
    assert status(visc=1, Re=0.0) == osbli.EINVAL
    # a valid configuration passes validation; with no workspace it stops at EWORKSPACE,
    # with one it reaches the device check (ECUDA on this GPU-less box, never a CPU fallback)
    p = osbli.make_params(n=(16, 16, 16), delta=(0.1, 0.1, 0.1))
    with pytest.raises(osbli.OsbliError) as e:
        osbli.osbli_init(p, 0, 0)
    assert e.value.status == osbli.EWORKSPACE
    with pytest.raises(osbli.OsbliError) as e:
        osbli.osbli_init(p, 4096 + 8, 1 << 40)
    assert e.value.status == osbli.EWORKSPACE                              # misaligned


def test_strerror(osbli):
    assert osbli.osbli_strerror(0) == "ok"
    assert "workspace" in osbli.osbli_strerror(osbli.EWORKSPACE)
    assert "unknown" in osbli.osbli_strerror(99)


def test_no_gpu_means_loud_failure_not_fallback(osbli):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = osbli.make_params(n=(16, 16, 16), delta=(0.1, 0.1, 0.1))
    with pytest.raises(osbli.OsbliError) as e:
        osbli.osbli_init(p, 4096, 1 << 40)
    assert e.value.status == osbli.ECUDA


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2007_14933_b200"
    bad = re.compile(r"^\s*(from|import)\s+oracle|libosbli_oracle|#\s*include\s*[\"<][^\n]*oracle|osbli_oracle\.", re.M)
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + list(pkg.rglob("*.h")):
        assert not bad.search(f.read_text()), f"{f} reaches into oracle/"
