"""CPU-side checks of the boundary: the library loads, exports every symbol include/tpc.h declares, and fails loudly without a GPU.
No compute call is made here."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def T():
    from paper_1905_05515_b200 import build
    build.build()
    import paper_1905_05515_b200 as T
    return T


def test_header_symbols_are_exported(T):
    hdr = open(os.path.join(ROOT, "include", "tpc.h")).read()
    declared = set(re.findall(r"^(?:int|void|const char\*)\s+(tpc_\w+)\s*\(", hdr, flags=re.M))
    assert declared == set(T.abi_symbols()), declared ^ set(T.abi_symbols())
    lib = T.load_library()
    for s in declared:
        assert getattr(lib, s) is not None
    assert lib.tpc_abi_version() == 1


def test_no_cpu_fallback(T):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(T.TpcError) as e:
        T.tpc_create(36, 152, np.linspace(85, 246, 152), 0.349, 250.0, 0.0, 0.1, 0.15, 0.5, 2.58)
    assert e.value.code == -4 and "no CPU fallback" in str(e.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1905_05515_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "tpc_oracle" not in src, f


def test_create_argument_errors_without_gpu(T):
    """Argument validation comes before the device check, so it is testable here: every bad geometry is TPC_E_ARG / TPC_E_CAPACITY."""
    rx = np.linspace(85, 246, 152)
    good = dict(n_sectors=36, n_rows=152, row_x=rx, sector_dphi=0.349, z_max=250.0, t_frame=0.0, sigma_y=0.1, sigma_z=0.15, bz=0.5,
                vdrift=2.58)
    def code(**kw):
        a = dict(good); a.update(kw)
        with pytest.raises(T.TpcError) as e:
            T.tpc_create(**a)
        return e.value.code
    bad_rx = rx.copy(); bad_rx[10] = bad_rx[9]
    assert code(row_x=bad_rx) == -1                       # not strictly increasing
    assert code(row_x=-rx) == -1                          # not positive
    assert code(n_sectors=0) == -1
    assert code(n_rows=2, row_x=rx[:2]) == -1
    assert code(n_rows=300, row_x=np.linspace(85, 246, 300)) == -5      # selector key holds 8 bits of row count
    assert code(bz=float("nan")) == -1 and code(vdrift=0.0) == -1 and code(vdrift=float("inf")) == -1
    assert code(sigma_y=0.0) == -1 and code(z_max=-1.0) == -1 and code(t_frame=-5.0) == -1 and code(sector_dphi=0.0) == -1
