"""CPU-side checks of the boundary (no compute calls): the C-ABI library builds, loads and exports
every symbol include/nsc.h declares; argument validation fails cleanly without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1908_00587_b200 import build, nsc
    build.build()
    return nsc.load_library()


def test_header_symbols_are_exported(lib):
    from paper_1908_00587_b200 import nsc
    hdr = open(os.path.join(ROOT, "include", "nsc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nsc_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations found in include/nsc.h"
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in nsc.h but not exported by libnsc.so"
    assert declared == set(nsc.EXPORTS)


def test_bad_arguments_are_rejected_before_touching_a_device(lib):
    from paper_1908_00587_b200 import nsc
    h = C.c_void_p()
    bad = [
        dict(N_r=8), dict(M_theta=0), dict(K_z=513), dict(K_z=8, n_z_phys=36), dict(eta=1.5), dict(alpha=-1.0),
        dict(k_theta0=0),
        dict(radial_grid=2), dict(Ra=10.0, Pr=0.0), dict(n_z_phys=20), dict(n_theta_phys=12),
    ]
    for over in bad:
        kw = dict(N_r=16, M_theta=8, K_z=8, eta=0.5, alpha=3.0, k_theta0=1, Re_i=1.0, Re_o=0.0, Ra=0.0, Pr=1.0,
                  radial_grid=1, n_theta_phys=0, n_z_phys=0, c=0.0, device=-1, radial_chunk=0)
        kw.update(over)
        p = nsc.nsc_params(**kw)
        assert lib.nsc_create_ex(C.byref(h), C.byref(p)) == nsc.NSC_EINVAL, over
        assert lib.nsc_last_error(None)
    assert lib.nsc_create_ex(None, None) == nsc.NSC_EINVAL
    assert lib.nsc_destroy(None) == nsc.NSC_OK
    assert lib.nsc_step(None, 1e-3) == nsc.NSC_EINVAL


def test_no_device_means_error_not_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1908_00587_b200 import nsc
    with pytest.raises(nsc.NscError) as ei:
        nsc.Context(16, 8, 8, 0.5, 3.0, 1, 100.0, 0.0)
    assert ei.value.code == nsc.NSC_ECUDA


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1908_00587_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                for line in open(os.path.join(dirpath, f)):
                    if re.match(r"\s*(import|from|#\s*include)\b", line):
                        assert "oracle" not in line, f"{f}: product code reaches into oracle/: {line!r}"
