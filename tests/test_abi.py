"""CPU-only checks of the boundary: the shared library builds/loads, exports every symbol the header declares,
and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def binding():
    from paper_2510_09812_b200 import build, binding
    build.build()
    return binding


def test_header_symbols_exported(binding):
    header = (ROOT / "include" / "cupymag_b200.h").read_text()
    declared = set(re.findall(r"^(?:int|const char \*)\s*(cm_\w+)\(", header, flags=re.M))
    assert len(declared) >= 20
    assert declared == set(binding.EXPORTS)
    L = C.CDLL(str(binding.LIB_PATH))
    for name in declared:
        assert hasattr(L, name), name
    assert b"sm_100a" in binding.lib().cm_version()


def test_struct_layouts_match_header(binding):
    # sizes implied by the header's field lists (x86-64 SysV)
    assert C.sizeof(binding.cm_material) == 8 * 8 + 9 * 8 + 8 + 8 + 9 * 8 + 6 * 8
    assert C.sizeof(binding.cm_step_params) == 8 + 24 + 4 + 4 + 8 + 4 + 4 + 4 + 4   # ... cg_precond, mech_matfree
    assert C.sizeof(binding.cm_step_info) == 4 * 10 + 8 * 10 + 24 + 8 + 8
    assert C.sizeof(binding.cm_profile) == 4 * 6 * 8


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2510_09812_b200 import inputs
    mesh = inputs.kuhn_box((3, 3, 3), (4e-9,) * 3)
    h = C.c_void_p()
    rc = binding.lib().cm_mesh_create(mesh.xyz.ctypes.data_as(C.c_void_p), mesh.n_nodes, mesh.tets.ctypes.data_as(C.c_void_p),
                                      mesh.n_tets, None, None, 1, None, C.byref(h))
    assert rc == binding.CM_E_CUDA
    assert b"no CUDA device" in binding.lib().cm_last_error()


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (nor through _work/)."""
    pkg = ROOT / "paper_2510_09812_b200"
    files = [f for ext in ("*.py", "*.cu", "*.h") for f in pkg.rglob(ext)]
    assert files
    for f in files:
        txt = f.read_text()
        assert "import oracle" not in txt and "from oracle" not in txt and "cm_oracle" not in txt, f
        assert "_work/" not in txt and "/_work" not in txt, f
    src = (ROOT / "oracle" / "cm_oracle.c").read_text()
    assert "cupymag_b200.h" not in src and "#include \"../" not in src
    py = (ROOT / "oracle" / "__init__.py").read_text()
    assert "import paper_2510_09812_b200" not in py and "from paper_2510_09812_b200" not in py


@pytest.mark.parametrize("axes", [1, 2, 5, 7])
def test_periodic_wrap_host_logic_matches_oracle(binding, oracle_mod, axes):
    """cm_periodic_wrap is host code (no device needed): bit-exact against the oracle's hash-map wrap."""
    import numpy as np
    from paper_2510_09812_b200 import inputs
    for grid, box in (((5, 4, 6), (20e-9, 12e-9, 25e-9)), ((33, 21, 17), (200e-9, 120e-9, 50e-9))):
        mesh = inputs.kuhn_box(grid, box, seed_mesh=3, seed_perm=4)
        dof, nd = binding.periodic_wrap(mesh.xyz, axes)
        dof_o, nd_o = oracle_mod.periodic_wrap(mesh.xyz, axes)
        assert nd == nd_o and np.array_equal(dof, dof_o)
    xyz = mesh.xyz.copy()
    i = np.flatnonzero((xyz[:, 0] == xyz[:, 0].max()) & (xyz[:, 1] > 0) & (xyz[:, 1] < xyz[:, 1].max()))[0]
    xyz[i, 1] += 1e-10
    with pytest.raises(binding.CmError) as ei:
        binding.periodic_wrap(xyz, 1)
    assert ei.value.code == binding.CM_E_BADARG
