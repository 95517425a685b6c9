"""cm_volume_average_noalloc against cm_volume_average (collected last on purpose: `pytest -x` stops at the first
failure, and this file tests an add-on outside the hot path, so it must not hide the parity tests).

The add-on exists for callers that cannot allocate device memory while they run: a host program whose own memory pool
already owns the whole device (a cudaMalloc inside the library would fail), or a time loop that reads <m> every step
while other streams are busy (a cudaMalloc / cudaFree may synchronise the whole device).  cm_volume_average grows a
staging buffer on demand; the add-on keeps its only scratch -- one partial sum per tile of 8192 nodes -- in a fixed
device array inside the library, shared by every call on the GPU and never cleared.  So the test makes two calls in a
row on one stream, the second one SMALLER than the first (fewer tiles, fewer components, another mesh), so that it
runs over the first call's left-overs, and checks both results against the existing path within the tolerance the
parity tests use for this quantity (tests/test_gpu_parity.py: 1e-13 fp64, 1e-7 fp32, absolute, on O(1) fields whose
weights sum to 1).  It needs nothing from the other test files and passes alone in a fresh process (where its first
call is the one that looks up the scratch address) as well as after them."""
import numpy as np
import pytest

from paper_2510_09812_b200 import inputs

pytestmark = pytest.mark.gpu

NM = 1e-9
TOL = {"f64": 1e-13, "f32": 1e-7}


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    return torch


@pytest.fixture(scope="module")
def cm():
    from paper_2510_09812_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def meshes(cm):
    """A: 50,061 nodes = 6 full tiles + a ragged one, Morton order (the gather through the permutation);
    B: 210 nodes = a single short tile, caller's order kept (no permutation)."""
    a = inputs.kuhn_box((41, 37, 33), (120 * NM, 108 * NM, 96 * NM), seed_mesh=71, seed_perm=72)
    b = inputs.kuhn_box((7, 6, 5), (18 * NM, 15 * NM, 12 * NM), seed_mesh=73, seed_perm=74)
    return ((a, cm.Mesh(a.xyz, a.tets, a.magnetic, a.elastic_id, cm.CM_REORDER_MORTON)),
            (b, cm.Mesh(b.xyz, b.tets, b.magnetic, b.elastic_id, cm.CM_REORDER_NONE)))


def _field(torch, n, nc, dtype, seed):
    g = np.random.default_rng(seed).normal(size=(n, nc) if nc > 1 else n)
    return torch.as_tensor(g, dtype=torch.float64 if dtype == "f64" else torch.float32, device="cuda")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_allocating_path(cm, torch, meshes, dtype):
    (ma, ga), (mb, gb) = meshes
    big = _field(torch, ma.n_nodes, 6, dtype, 1)       # 7 tiles x 6 components: fills 42 words of the scratch
    small = _field(torch, mb.n_nodes, 3, dtype, 2)     # then 1 tile x 3 components over the same words
    one = _field(torch, ma.n_nodes, 1, dtype, 3)
    out_big = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    out_small = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    out_one = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    # back to back on one stream, no synchronisation in between: stream order is what keeps them apart
    ga.volume_average_noalloc(big, out_big)
    gb.volume_average_noalloc(small, out_small)
    ga.volume_average_noalloc(one, out_one)
    torch.cuda.synchronize()
    got = [out_big.cpu().numpy(), out_small.cpu().numpy(), out_one.cpu().numpy()]
    want = [ga.volume_average(big), gb.volume_average(small), ga.volume_average(one)]
    for g, w in zip(got, want):
        assert np.isfinite(g).all()
        assert np.abs(g - w).max() <= TOL[dtype]
    # the same three calls again: same bits (fixed summation order, nothing left over from the calls before matters),
    # and the device's free memory does not move (every kernel is loaded by now, the outputs exist already)
    again = [torch.empty_like(out_big), torch.empty_like(out_small), torch.empty_like(out_one)]
    free0 = torch.cuda.mem_get_info()[0]
    ga.volume_average_noalloc(big, again[0])
    gb.volume_average_noalloc(small, again[1])
    ga.volume_average_noalloc(one, again[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    for g, a in zip(got, again):
        assert np.array_equal(g, a.cpu().numpy())


def test_sizes_beyond_the_fixed_scratch_are_refused(cm, torch, meshes):
    (ma, ga), _ = meshes
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    with pytest.raises(cm.CmError) as ei:
        ga.volume_average_noalloc(_field(torch, ma.n_nodes, 2, "f64", 4), out)
    assert ei.value.code == cm.CM_E_BADARG and "1, 3 or 6" in str(ei.value)
    torch.cuda.synchronize()
    assert (out == 0).all()                            # nothing was launched
    assert cm.CM_NOALLOC_MAX_NODES == 2048 * 8192      # the stated limit: 2048 scratch rows, one per tile of 8192 nodes
