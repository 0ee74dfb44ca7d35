"""The five BASELINE.json configurations as seeded synthetic blocks (DATA ONLY, no method
arithmetic).  A block = dict(shape, P, lam, deformed, v0, E, seed): an affine sub-map per element
(v0, E) optionally composed with the sinusoidal map of config 2; geometric factors are produced by
workloads.synthetic from the quadrature-point coordinates `xi` that the caller supplies.
Recipe and citations: DESIGN.md section 6."""
import torch

from . import synthetic as wl

HEX, TET, PRISM = 0, 1, 2


def _slab(mesh_fn, n, zlo, zhi, device):
    return mesh_fn(n, zlo, zhi, device=device)


def config_blocks(cfg, device="cpu", P_sweep=None, scale=1.0):
    """Returns (name, op, blocks).  `scale` < 1 shrinks the mesh (tests); 1.0 = BASELINE sizes."""
    seed = wl.SEED0 + cfg
    if cfg == 1:
        v0, E = wl.hex_mesh(4, device=device)
        return "cfg1 hex affine P3 Q5, 64 el", "helmholtz", [dict(shape=HEX, P=3, lam=1.0, deformed=False, v0=v0, E=E, seed=seed)]
    if cfg == 2:
        # P_sweep: the same workload at another order, cube count chosen to keep the DoF of the P=4 case
        P = 4 if P_sweep is None else P_sweep
        n0 = 32 if P == 4 else (32 ** 3 * 125.0 / (P + 1) ** 3) ** (1.0 / 3.0)
        n = max(2, int(round(n0 * scale)))
        v0, E = wl.hex_mesh(n, device=device)
        return ("cfg2 hex deformed P%d Q%d, %d^3 el" % (P, P + 2, n), "helmholtz",
                [dict(shape=HEX, P=P, lam=1.0, deformed=True, v0=v0, E=E, seed=seed)])
    if cfg == 3:
        P = 4 if P_sweep is None else P_sweep
        n0 = 32 if P == 4 else (32 ** 3 * 35.0 * 6 / ((P + 1) * (P + 2) * (P + 3))) ** (1.0 / 3.0)
        n = max(2, int(round(n0 * scale)))
        v0, E = wl.kuhn_tet_mesh(n, device=device)
        return ("cfg3 tet affine P%d Q%d, 6x%d^3 el" % (P, P + 2, n), "helmholtz",
                [dict(shape=TET, P=P, lam=1.0, deformed=False, v0=v0, E=E, seed=seed)])
    if cfg == 4:
        P_sweep = 4 if P_sweep is None else P_sweep
        n = max(2, int(round(wl.p_sweep_cubes(P_sweep) * scale)))
        v0, E = wl.hex_mesh(n, device=device)
        return ("cfg4 hex affine P%d Q%d, %d^3 el" % (P_sweep, P_sweep + 2, n), "mass+laplacian",
                [dict(shape=HEX, P=P_sweep, lam=0.0, deformed=False, v0=v0, E=E, seed=seed)])
    if cfg == 5:
        P = 5 if P_sweep is None else P_sweep
        # other orders: cube count chosen to keep the geometry stream of the P=5 case (3.7 GB)
        n0 = 40 if P == 5 else 40 * 7.0 / (P + 2)
        n = max(4, int(round(n0 * scale)))
        zt = max(1, n // 4)                       # z-layers 0..n/4-1 -> tets, the rest -> prisms
        vt, Et = wl.kuhn_tet_mesh(n, 0, zt, device=device)
        vp, Ep = wl.prism_mesh(n, zt, n, device=device)
        return ("cfg5 hybrid deformed P%d Q%d, %d tets + %d prisms" % (P, P + 2, vt.shape[0], vp.shape[0]), "helmholtz",
                [dict(shape=PRISM, P=P, lam=10.0, deformed=True, v0=vp, E=Ep, seed=seed),
                 dict(shape=TET, P=P, lam=10.0, deformed=True, v0=vt, E=Et, seed=seed + 100)])
    raise ValueError("config 1..5")


def block_factors(block, xi, chunk=4096):
    """(dxi_dx, detJ) of a block on the device of its mesh; xi [Nq][3] from the caller."""
    if block["deformed"]:
        return wl.sinusoidal_factors(block["v0"], block["E"], xi.to(block["v0"].device), chunk=chunk)
    return wl.affine_factors(block["v0"], block["E"])


def shard(block, rank, world):
    """Contiguous element range of `block` for `rank` (elements are independent: P:163)."""
    ne = block["v0"].shape[0]
    lo, hi = ne * rank // world, ne * (rank + 1) // world
    out = dict(block)
    out["v0"], out["E"] = block["v0"][lo:hi].contiguous(), block["E"][lo:hi].contiguous()
    out["range"] = (lo, hi)
    return out
