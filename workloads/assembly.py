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


def partition_l2g(l2g, nglobal, world):
    """Splits a mesh with local-to-global map `l2g` [nelem][nm] into `world` contiguous element ranges (the shards of
    workloads.configs.shard) and describes each rank's share of the global system (DATA ONLY: integer bookkeeping).

    Returns one dict per rank:
      range          (lo, hi) element range
      glob           int64 [nr]: global dof of every rank-local dof, ascending (the rank's numbering)
      l2g            int64 [hi-lo][nm]: the rank's map in its own numbering
      shared_dof     int64 [ns]: rank-local dofs that other ranks hold too (the interface), ascending
      shared_slot    int64 [ns]: their position in the interface vector, the same on every rank
      shared_mult    int32 [ns]: number of ranks that hold each of them (>= 2)
      n_interface    length of the interface vector (dofs held by more than one rank)
    """
    nelem = l2g.shape[0]
    bounds = [nelem * r // world for r in range(world + 1)]
    held = torch.zeros(nglobal, dtype=torch.int32)
    globs = []
    for r in range(world):
        g = torch.unique(l2g[bounds[r]:bounds[r + 1]].reshape(-1))      # sorted
        globs.append(g)
        held[g] += 1
    iface = torch.nonzero(held > 1).reshape(-1)                         # ascending global ids
    slot_of = torch.full((nglobal,), -1, dtype=torch.int64)
    slot_of[iface] = torch.arange(iface.numel(), dtype=torch.int64)
    parts = []
    for r in range(world):
        g = globs[r]
        loc_of = torch.full((nglobal,), -1, dtype=torch.int64)
        loc_of[g] = torch.arange(g.numel(), dtype=torch.int64)
        sh = torch.nonzero(held[g] > 1).reshape(-1)
        parts.append(dict(range=(bounds[r], bounds[r + 1]), glob=g.contiguous(),
                          l2g=loc_of[l2g[bounds[r]:bounds[r + 1]]].contiguous(),
                          shared_dof=sh.to(torch.int64).contiguous(), shared_slot=slot_of[g[sh]].contiguous(),
                          shared_mult=held[g[sh]].to(torch.int32).contiguous(), n_interface=int(iface.numel())))
    return parts
