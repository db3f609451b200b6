"""The C-ABI library loads and exports every symbol include/sph.h declares (no compute, no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2512_09904_b200 import build
    return build.build_library()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_]+)\s*\(", src)))


def test_header_declares_the_six_calls():
    names = declared_functions()
    for f in ("sph_create", "sph_load_particles", "sph_set_gear_kinematics", "sph_step", "sph_get_fields",
              "sph_get_torque", "sph_destroy"):
        assert f in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for f in declared_functions():
        assert hasattr(L, f), f


def test_params_struct_matches_header_size(libpath):
    """sph_create checks struct_size; a wrong ctypes mirror is caught here without a GPU: create must
    fail with SPH_EINVAL for a bad size, and with SPH_ECUDA (no device) or succeed for the right one."""
    from paper_2512_09904_b200 import api, workloads as wl
    w = wl.still_tank(n=4)
    p = api.make_params(w.params, w.bodies)
    ctx = ctypes.c_void_p()
    p.struct_size += 8
    assert api.lib().sph_create(ctypes.byref(p), ctypes.byref(ctx)) == api.SPH_EINVAL
    p.struct_size -= 8
    rc = api.lib().sph_create(ctypes.byref(p), ctypes.byref(ctx))
    assert rc in (api.SPH_OK, api.SPH_ECUDA), api.lib().sph_last_error(None)
    if rc == api.SPH_OK:
        api.sph_destroy(ctx)
    else:
        assert b"no CPU fallback" in api.lib().sph_last_error(None)


def test_no_product_import_of_oracle():
    """the product path never imports, links or reads oracle/."""
    pkg = os.path.join(ROOT, "paper_2512_09904_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "sph_oracle" not in txt, f
