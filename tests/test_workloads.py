"""Checks of the seeded synthetic-input generators (data only)."""
import math

import numpy as np
import pytest
import torch

from oracle import nk_oracle as o
from workloads import synthetic as S


def test_coefficients_seeded_uniform():
    a = S.coefficients(S.SEED0 + 1, 64, 64)
    b = S.coefficients(S.SEED0 + 1, 64, 64)
    assert a.dtype == torch.float64 and torch.equal(a, b)
    assert a.min() >= -1 and a.max() <= 1 and abs(a.mean().item()) < 0.05
    assert not torch.equal(a, S.coefficients(S.SEED0 + 2, 64, 64))


def test_config4_cube_counts():
    assert [S.p_sweep_cubes(P) for P in range(1, 11)] == [184, 123, 92, 74, 61, 53, 46, 41, 37, 33]


@pytest.mark.parametrize("mesh,shape,per_cube", [(S.hex_mesh, o.HEX, 1), (S.kuhn_tet_mesh, o.TET, 6), (S.prism_mesh, o.PRISM, 2)])
def test_meshes_tile_the_unit_cube(mesh, shape, per_cube):
    n = 3
    v0, E = mesh(n)
    assert v0.shape[0] == per_cube * n ** 3
    el = o.Element(shape, 2, 4)
    A, J = S.affine_factors(v0, E)
    assert J.min() > 0
    vol = el.wq.sum() * J[:, 0]
    assert vol.sum().item() == pytest.approx(1.0, rel=1e-13)
    np.testing.assert_allclose(vol.numpy(), 1.0 / (per_cube * n ** 3), rtol=1e-13)
    # all mapped quadrature points lie in the unit cube; element centroids are distinct
    X = v0[:, None, :] + torch.einsum("eab,nb->ena", 0.5 * E, torch.tensor(el.xi) + 1.0)
    assert X.min() >= -1e-14 and X.max() <= 1 + 1e-14
    cent = (X * torch.tensor(el.wq)[None, :, None]).sum(1) / el.wq.sum()
    assert len({tuple(np.round(c, 9)) for c in cent.numpy()}) == v0.shape[0]


@pytest.mark.parametrize("mesh,shape", [(S.hex_mesh, o.HEX), (S.kuhn_tet_mesh, o.TET), (S.prism_mesh, o.PRISM)])
def test_sinusoidal_factors_are_the_inverse_jacobian(mesh, shape):
    n = 2
    v0, E = mesh(n)
    el = o.Element(shape, 3, 5)
    xi = torch.tensor(el.xi)
    A, J = S.sinusoidal_factors(v0, E, xi, chunk=5)
    assert A.shape == (v0.shape[0], el.Nq, 3, 3) and J.shape == (v0.shape[0], el.Nq)

    def X(xi_):
        x = v0[:, None, :] + torch.einsum("eab,enb->ena", 0.5 * E, xi_ + 1.0)
        return S.sinusoidal_map(x)
    base = xi[None].expand(v0.shape[0], -1, -1)
    h = 1e-6
    dX = torch.stack([(X(base + h * torch.eye(3, dtype=torch.float64)[a]) - X(base - h * torch.eye(3, dtype=torch.float64)[a])) / (2 * h)
                      for a in range(3)], dim=-1)                 # [e][n][c][a] = dX_c/dxi_a
    np.testing.assert_allclose(torch.einsum("enjc,enca->enja", A, dX).numpy(),
                               np.broadcast_to(np.eye(3), A.shape), atol=1e-8)
    np.testing.assert_allclose(J.numpy(), torch.linalg.det(dX).numpy(), rtol=1e-8)
    assert J.min() > 0
    # the map sends the unit cube onto itself: total volume 1 (quadrature error only)
    assert (J * torch.tensor(el.wq)).sum().item() == pytest.approx(1.0, abs=1e-3)


def test_sinusoidal_det_range():
    x = torch.rand(20000, 3, dtype=torch.float64)
    tp = 2 * math.pi
    g = tp * (torch.cos(tp * x[:, 0]) * torch.sin(tp * x[:, 1]) * torch.sin(tp * x[:, 2])
              + torch.sin(tp * x[:, 0]) * torch.cos(tp * x[:, 1]) * torch.sin(tp * x[:, 2])
              + torch.sin(tp * x[:, 0]) * torch.sin(tp * x[:, 1]) * torch.cos(tp * x[:, 2]))
    d = 1 + 0.05 * g
    assert d.min() > 0.63 and d.max() < 1.37
