"""Connectivity of the structured hex meshes of workloads.synthetic (DATA ONLY: integer maps, no method arithmetic).

hex_l2g(n, P): the local-to-global map of the C0 modified basis (A7) on the n^3 cubes of hex_mesh(n),
element index ix + n*(iy + n*iz), local mode (p,q,r) at storage rank (p*nm + q)*nm + r (A3) with p, q, r running
along x, y, z.  Along one direction a 1-D element e owns the modes a = 0 (left vertex), a = 1 (right vertex) and
a >= 2 (interior); their global 1-D indices are e*P, (e+1)*P and e*P + a - 1, so that neighbouring elements share
their vertex and nothing else, and the 3-D global dof is the tensor product (gx*N1 + gy)*N1 + gz, N1 = n*P + 1.
All elements have the same orientation, so shared edge and face modes need no sign flip.
"""
import torch


def hex_l2g(n, P):
    """returns (l2g int64 [n^3][(P+1)^3], nglobal)"""
    nm, N1 = P + 1, n * P + 1
    a = torch.arange(nm)
    off = torch.where(a == 0, torch.zeros_like(a), torch.where(a == 1, torch.full_like(a, P), a - 1))   # [nm]
    e = torch.arange(n)
    g1 = e[:, None] * P + off[None, :]                       # [n][nm] global 1-D index of mode a of 1-D element e
    gx = g1[None, None, :, :, None, None]                    # [iz][iy][ix][p][q][r]
    gy = g1[None, :, None, None, :, None]
    gz = g1[:, None, None, None, None, :]
    l2g = (gx * N1 + gy) * N1 + gz
    l2g = l2g.expand(n, n, n, nm, nm, nm).reshape(n ** 3, nm ** 3).contiguous().to(torch.int64)
    return l2g, N1 ** 3


def hex_boundary_dofs(n, P):
    """global dofs of hex_l2g(n, P) that lie on the boundary of the unit cube (a 1-D index 0 or n*P in any direction):
    int64 tensor, ascending"""
    N1 = n * P + 1
    g = torch.arange(N1)
    on = (g == 0) | (g == N1 - 1)
    m = on[:, None, None] | on[None, :, None] | on[None, None, :]
    return torch.nonzero(m.reshape(-1)).reshape(-1).to(torch.int64).contiguous()
