"""CPU-side checks of the boundary: librad.so builds, loads and exports every symbol include/rad.h declares;
the binding marshals without a GPU; the product path has no CPU fallback."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def so():
    from paper_2302_04283_b200 import build
    return build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "rad.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rad_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_survey_entry_points():
    names = declared_functions()
    for must in ("rad_create", "rad_stage", "rad_moments", "rad_destroy", "rad_get_table", "rad_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(so):
    lib = ctypes.CDLL(so)
    for name in declared_functions():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_names(so):
    from paper_2302_04283_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()
    for name in binding.EXPORTS:
        assert hasattr(binding, name) or name in ("rad_last_error",)


def test_header_is_plain_c(tmp_path):
    """the header compiles as C99 (no C++ or torch types in the signatures)"""
    import subprocess
    f = tmp_path / "t.c"
    f.write_text('#include "rad.h"\nint main(void){ rad_params p; (void)p; return RAD_OK; }\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), "-c", str(f), "-o", str(tmp_path / "t.o")])


def test_no_gpu_means_error_not_fallback(so):
    """without a CUDA device rad_create must fail with RAD_ECUDA; argument errors are reported before that"""
    import torch
    from paper_2302_04283_b200 import binding as B
    grid = dict(n=(4, 4, 4), x0=(0, 0, 0), dx=(1, 1, 1))
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), dict(grid, ng=1), ("latlon", 2, 4), None, dict(couple=0))
    assert e.value.status == 1  # RAD_EINVAL: ng must be 2 or 3
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("geodesic", 2), None, dict(couple=0, recon_angle=1))
    assert e.value.status == 4  # RAD_EUNSUPPORTED: PLM in angle is for lat-lon grids (MAPR is not implemented)
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("latlon", 2, 5), None, dict(couple=0, recon_angle=1))
    assert e.value.status == 4  # ... with even npsi (the pole-crossing stencil)
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("latlon", 2, 4), None, dict(couple=0, recon_space=2))
    assert e.value.status == 1  # PPM needs ng = 3
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), dict(grid, bc_hi=(4, 0, 0)), ("latlon", 2, 4), None, dict(couple=0))
    assert e.value.status == 1  # bad boundary code
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("latlon", 2, 4), None, dict(couple=0, tau_factor=1.0))
    assert e.value.status == 1  # RAD_EINVAL: the optical-depth-aware flux (Eq.26-29) needs opacities
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("latlon", 2, 4), None, dict(couple=0, tau_factor=-1.0))
    assert e.value.status == 1
    with pytest.raises(B.RadError) as e:
        B.rad_create(dict(kind=0), grid, ("latlon", 2, 4), None, dict(couple=1))
    assert e.value.status == 1  # coupling needs opacities
    if not torch.cuda.is_available():
        with pytest.raises(B.RadError) as e:
            B.rad_create(dict(kind=0), grid, ("latlon", 2, 4), None, dict(couple=0))
        assert e.value.status == 3  # RAD_ECUDA


def test_product_does_not_import_the_oracle():
    """the CUDA package never references oracle/ (and the oracle never references the package)"""
    pkg = os.path.join(ROOT, "paper_2302_04283_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "rad_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2302_04283_b200" not in txt.replace("paper_2302_04283_b200/csrc (the CUDA path)", "") and "librad.so" not in txt, f
