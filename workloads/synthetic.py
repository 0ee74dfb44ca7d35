"""Seeded, synthetic inputs shaped like the paper's workloads (P:364-384:
Helmholtz on blocks of like hex / tet elements, a range of orders, up to ~1e8
DoF).  They stand in for the Nektar++ meshes of the paper, which are not
available here.  DATA ONLY: random coefficients and closed-form geometric
factors; none of the method's arithmetic (bases, quadrature, contractions)
lives here.  The standard-element coordinates `xi` of the quadrature points
are an INPUT (each side supplies its own).

Every element is an affine image of the standard element,
    x(xi) = v0 + E (xi + 1)/2,   E = [a b c] (columns = edge vectors),
optionally composed with the global map X = x + amp*s(x)*(1,1,1)^T,
s = sin(2 pi x) sin(2 pi y) sin(2 pi z) (config 2 / config 5).
Outputs follow the C-ABI convention (include/nk.h): dxi_dx[e][n][j][i] =
d xi_j / d X_i, detJ[e][n] > 0, n = 1 point if affine, Nq if deformed.
"""
import itertools
import math

import numpy as np
import torch

SEED0 = 20917
F64 = torch.float64


def coefficients(seed, nelem, nm, device="cpu"):
    """i.i.d. uniform[-1,1] fp64, element-major [nelem][nm] (Philox stream)."""
    rng = np.random.Generator(np.random.Philox(seed))
    a = rng.random((nelem, nm)) * 2.0 - 1.0
    return torch.from_numpy(a).to(device)


def point_values(seed, nelem, nq, ncomp=1, device="cpu"):
    rng = np.random.Generator(np.random.Philox(seed))
    a = rng.random((ncomp, nelem, nq)) * 2.0 - 1.0
    t = torch.from_numpy(a).to(device)
    return t[0] if ncomp == 1 else t


# ----------------------------------------------------------------------------
# meshes: (v0 [ne,3], E [ne,3,3]) per element
# ----------------------------------------------------------------------------
def _cube_corners(n, zlo=0, zhi=None, device="cpu"):
    zhi = n if zhi is None else zhi
    h = 1.0 / n
    iz, iy, ix = torch.meshgrid(torch.arange(zlo, zhi, device=device),
                                torch.arange(n, device=device),
                                torch.arange(n, device=device), indexing="ij")
    c = torch.stack([ix.reshape(-1), iy.reshape(-1), iz.reshape(-1)], dim=1).to(F64) * h
    return c, h


def hex_mesh(n, device="cpu"):
    """n^3 cubes of the unit cube, element index ix + n*(iy + n*iz)."""
    c, h = _cube_corners(n, device=device)
    E = (h * torch.eye(3, dtype=F64, device=device)).expand(c.shape[0], 3, 3).contiguous()
    return c, E


def kuhn_tet_mesh(n, zlo=0, zhi=None, device="cpu"):
    """Each cube -> 6 Kuhn tets (one per permutation of the axes); element
    index 6*cube + t.  v1 = v0 + h e_pi0, v2 = v1 + h e_pi1, v3 = v2 + h e_pi2,
    v2 and v3 swapped when the orientation is negative."""
    c, h = _cube_corners(n, zlo, zhi, device=device)
    eye = np.eye(3)
    Es = []
    for perm in itertools.permutations(range(3)):
        d1 = eye[perm[0]]
        d2 = d1 + eye[perm[1]]
        d3 = d2 + eye[perm[2]]
        E = np.stack([d1, d2, d3], axis=1)           # columns v_j - v0
        if np.linalg.det(E) < 0:
            E = np.stack([d1, d3, d2], axis=1)
        Es.append(h * E)
    Es = torch.tensor(np.stack(Es), dtype=F64, device=device)    # [6,3,3]
    ne = c.shape[0]
    v0 = c[:, None, :].expand(ne, 6, 3).reshape(-1, 3).contiguous()
    E = Es[None].expand(ne, 6, 3, 3).reshape(-1, 3, 3).contiguous()
    return v0, E


def prism_mesh(n, zlo=0, zhi=None, device="cpu"):
    """Each cube -> 2 prisms cut along the x-z diagonal, triangle spanned by
    (a,c), extruded along b; element index 2*cube + t."""
    c, h = _cube_corners(n, zlo, zhi, device=device)
    ex, ey, ez = (torch.tensor(v, dtype=F64, device=device) for v in
                  ([1., 0, 0], [0, 1., 0], [0, 0, 1.]))
    Elo = h * torch.stack([ex, ey, ez], dim=1)
    Eup = h * torch.stack([-ex, ey, -ez], dim=1)
    ne = c.shape[0]
    v0 = torch.stack([c, c + h * (ex + ez)], dim=1).reshape(-1, 3).contiguous()
    E = torch.stack([Elo, Eup])[None].expand(ne, 2, 3, 3).reshape(-1, 3, 3).contiguous()
    return v0, E


# ----------------------------------------------------------------------------
# geometric factors
# ----------------------------------------------------------------------------
def _inv3_det3(M):
    """Inverse and determinant of a batch of 3x3 matrices [..., 3, 3] by cofactors: elementwise arithmetic only.
    No library routine (batched LU, GEMM) on purpose: on the GPU those may pick another algorithm from one process
    to the next, and a full-size parity test then fails on its INPUTS (seen on B200: the first elements of config 2
    2e-10 away from the host evaluation in one run out of five when the factors went through einsum / linalg)."""
    a, b, c = M[..., 0, 0], M[..., 0, 1], M[..., 0, 2]
    d, e, f = M[..., 1, 0], M[..., 1, 1], M[..., 1, 2]
    g, h, i = M[..., 2, 0], M[..., 2, 1], M[..., 2, 2]
    c00, c01, c02 = e * i - f * h, f * g - d * i, d * h - e * g
    det = a * c00 + b * c01 + c * c02
    adj = torch.stack([torch.stack([c00, c * h - b * i, b * f - c * e], dim=-1),
                       torch.stack([c01, a * i - c * g, c * d - a * f], dim=-1),
                       torch.stack([c02, b * g - a * h, a * e - b * d], dim=-1)], dim=-2)
    return adj / det[..., None, None], det


def affine_factors(v0, E):
    """dxi_dx [ne][1][3][3] = (E/2)^-1, detJ [ne][1] = |det(E/2)|."""
    inv, det = _inv3_det3(0.5 * E)
    return inv[:, None].contiguous(), det.abs()[:, None].contiguous()


def sinusoidal_factors(v0, E, xi, amp=0.05, chunk=4096):
    """Analytic factors of X = x + amp*s(x)*(1,1,1)^T composed with the affine
    sub-map, at the points xi [Nq][3]:  F = I + amp*1 grad(s)^T,
    det F = 1 + amp*(s_x+s_y+s_z),  F^-1 = I - amp*1 grad(s)^T / det F,
    dxi/dX = (E/2)^-1 F^-1,  detJ = |det(E/2)| det F."""
    dev = v0.device
    xi = torch.as_tensor(xi, dtype=F64, device=dev)
    ne, nq = v0.shape[0], xi.shape[0]
    A = torch.empty((ne, nq, 3, 3), dtype=F64, device=dev)
    J = torch.empty((ne, nq), dtype=F64, device=dev)
    tp = 2.0 * math.pi
    ones = torch.ones(3, dtype=F64, device=dev)
    for s0 in range(0, ne, chunk):
        sl = slice(s0, min(ne, s0 + chunk))
        Jm = 0.5 * E[sl]
        Ainv, detA = _inv3_det3(Jm)                                  # [c,3,3], [c]
        x = v0[sl, None, :] + (Jm[:, None, :, :] * (xi + 1.0)[None, :, None, :]).sum(-1)      # [c,n,3]
        sn, cs = torch.sin(tp * x), torch.cos(tp * x)
        g = tp * torch.stack([cs[..., 0] * sn[..., 1] * sn[..., 2],
                              sn[..., 0] * cs[..., 1] * sn[..., 2],
                              sn[..., 0] * sn[..., 1] * cs[..., 2]], dim=-1)   # grad s
        detF = 1.0 + amp * g.sum(-1)
        Finv = torch.eye(3, dtype=F64, device=dev) - amp * ones[:, None] * g[..., None, :] / detF[..., None, None]
        A[sl] = (Ainv[:, None, :, :, None] * Finv[:, :, None, :, :]).sum(-2)                  # A_jk Finv_ki
        J[sl] = detA.abs()[:, None] * detF
    return A, J


def sinusoidal_map(x, amp=0.05):
    """The global map itself (for tests of the generator)."""
    s = torch.sin(2 * math.pi * x).prod(-1, keepdim=True)
    return x + amp * s


def p_sweep_cubes(P):
    """Config 4: cubes per side so that n^3 (P+1)^3 ~ 5e7 DoF."""
    return int(round((5e7 / (P + 1) ** 3) ** (1.0 / 3.0)))
