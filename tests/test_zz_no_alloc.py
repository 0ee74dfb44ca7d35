"""nk_assembled_helmholtz_apply_static (include/nk.h): the assembled Helmholtz apply with its work space in the library's
static device array, for callers that cannot allocate.  Checked against the existing path (nk_assembled_helmholtz_apply,
itself checked against the oracle's assembled matrix in test_gpu_solver.py) on calls in a row that share the array.
Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

import nk_cases as K
from oracle import nk_oracle as o
from workloads import assembly as asm

pytestmark = pytest.mark.gpu
TOL = 1e-12          # the normwise tolerance of the parity tests (A18)


@pytest.fixture(scope="module")
def nk():
    import paper_2606_20917_b200 as nk
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return nk


def block(nk, n, P, deformed):
    A, J = K.geometry(o.HEX, P, n, deformed)
    basis = nk.Basis(o.HEX, P)
    geom = nk.Geom(basis, A.cuda(), J.cuda(), deformed)
    l2g, ng = asm.hex_l2g(n, P)
    return basis, geom, nk.GatherScatter(l2g, ng), ng


def both(nk, blk, lam, u):
    basis, geom, gs, ng = blk
    ref = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
    got = torch.full((ng,), float("nan"), dtype=torch.float64, device="cuda")
    nk.assembled_helmholtz_apply(basis, geom, gs, lam, u, ref)
    nk.assembled_helmholtz_apply_static(basis, geom, gs, lam, u, got)
    torch.cuda.synchronize()
    return got.cpu().numpy(), ref.cpu().numpy()


def test_static_apply_matches_existing_path_on_calls_in_a_row(nk):
    lam = 1.75
    big, small = block(nk, 4, 4, True), block(nk, 2, 3, True)      # 8000 and 512 local dofs, deformed hexes
    rng = np.random.Generator(np.random.Philox(2606))
    for blk in (big, big, small, big):                             # the small call runs on what the big one left behind
        u = torch.from_numpy(rng.standard_normal(blk[3])).cuda()
        got, ref = both(nk, blk, lam, u)
        assert np.isfinite(ref).all() and np.abs(ref).max() > 0
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
        assert np.array_equal(got, ref)                            # same kernels, same order of sums
    # constrained dofs go through the same two kernels
    basis, geom, gs, ng = big
    gs.set_constrained(asm.hex_boundary_dofs(4, 4))
    got, ref = both(nk, big, 0.0, torch.from_numpy(rng.standard_normal(ng)).cuda())
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_static_apply_allocates_no_device_memory(nk):
    blk = block(nk, 3, 4, True)
    basis, geom, gs, ng = blk
    u = torch.randn(ng, dtype=torch.float64, device="cuda")
    out = torch.empty_like(u)
    nk.assembled_helmholtz_apply_static(basis, geom, gs, 1.0, u, out)      # warm: module load, occupancy cache
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        nk.assembled_helmholtz_apply_static(basis, geom, gs, 1.0, u, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_apply_rejects_what_it_cannot_serve(nk):
    limit = nk.static_max_local_dofs()
    assert limit == 1048576
    # beyond the limit: 51^3 trilinear hexes = 1061208 local dofs
    n = 51
    assert n ** 3 * 8 > limit
    blk = block(nk, n, 1, False)
    basis, geom, gs, ng = blk
    u = torch.ones(ng, dtype=torch.float64, device="cuda")
    out = torch.full_like(u, 7.0)
    with pytest.raises(nk.NkError) as ei:
        nk.assembled_helmholtz_apply_static(basis, geom, gs, 1.0, u, out)
    assert "NK_STATIC_MAX_LOCAL_DOFS" in str(ei.value) and "1061208" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                 # nothing was launched
    # an affine block on the reference-matrix form (trilinear hexes) before its matrices are resident: refused, then
    # served once nk_helmholtz_apply has run on the block
    blk = block(nk, 4, 1, False)
    basis, geom, gs, ng = blk
    if nk.get_affine_simplex_form() != 1:
        u = torch.from_numpy(np.random.Generator(np.random.Philox(5)).standard_normal(ng)).cuda()
        with pytest.raises(nk.NkError) as ei:
            nk.assembled_helmholtz_apply_static(basis, geom, gs, 1.0, u, torch.empty_like(u))
        assert "set-up" in str(ei.value)
        loc = torch.zeros(4 ** 3 * 8, dtype=torch.float64, device="cuda")
        nk.helmholtz_apply(basis, geom, 1.0, loc, torch.empty_like(loc))
        got, ref = both(nk, blk, 1.0, u)
        assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
