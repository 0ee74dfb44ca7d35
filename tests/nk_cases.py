"""Shared helpers of the GPU parity tests: seeded cases shaped like BASELINE.json's configs, the
error metric of DESIGN.md A18, and thin wrappers that run one operator through the C-ABI binding.
Test infrastructure: may import oracle/; the product package never does."""
import numpy as np
import torch

from oracle import nk_oracle as o
from workloads import synthetic as wl

_ELS = {}


def element(shape, P, Q=None):
    Q = P + 2 if Q is None else Q
    key = (shape, P, Q)
    if key not in _ELS:
        _ELS[key] = o.Element(shape, P, Q)
    return _ELS[key]


def mesh(shape, n, zlo=0, zhi=None):
    if shape == o.HEX:
        c, E = wl.hex_mesh(n)
        if zlo or zhi is not None:
            zhi = n if zhi is None else zhi
            sl = slice(zlo * n * n, zhi * n * n)
            c, E = c[sl], E[sl]
        return c, E
    if shape == o.TET:
        return wl.kuhn_tet_mesh(n, zlo, zhi)
    return wl.prism_mesh(n, zlo, zhi)


def geometry(shape, P, n, deformed, take=None, zlo=0, zhi=None, xi=None):
    """(dxi_dx [ne][npt][3][3], detJ [ne][npt]) as CPU fp64 tensors."""
    v0, E = mesh(shape, n, zlo, zhi)
    if take is not None:
        v0, E = v0[take].contiguous(), E[take].contiguous()
    if deformed:
        xi = element(shape, P).xi if xi is None else xi
        return wl.sinusoidal_factors(v0, E, xi)
    return wl.affine_factors(v0, E)


def normwise_err(got, ref):
    """A18: per element max|got-ref| / max|ref|, then the max over elements."""
    got = np.asarray(got, dtype=np.float64).reshape(ref.shape[0], -1)
    ref = np.asarray(ref, dtype=np.float64).reshape(ref.shape[0], -1)
    den = np.abs(ref).max(axis=1)
    den[den == 0] = 1.0
    return float((np.abs(got - ref).max(axis=1) / den).max()) if ref.size else 0.0


OPS = ("bwdtrans", "iprod", "physderiv", "iprod_deriv", "mass", "laplacian", "helmholtz")


def oracle_op(op, el, A, J, lam, x):
    """x: numpy input ([ne][Nm], [ne][Nq] or [3][ne][Nq]); returns numpy output."""
    A, J = A.numpy(), J.numpy()
    if op == "bwdtrans":
        return o.bwdtrans(el, x)
    if op == "iprod":
        return o.iprod(el, J, x)
    if op == "physderiv":
        return o.physderiv(el, A, x)
    if op == "iprod_deriv":
        return o.iprod_deriv(el, A, J, x)
    if op == "mass":
        return o.mass(el, J, x)
    if op == "laplacian":
        return o.laplacian(el, A, J, x)
    if op == "helmholtz":
        return o.helmholtz(el, A, J, lam, x)
    raise KeyError(op)


def make_input(op, seed, ne, el):
    if op in ("bwdtrans", "mass", "laplacian", "helmholtz"):
        return wl.coefficients(seed, ne, el.Nm).numpy()
    if op in ("iprod", "physderiv"):
        return wl.point_values(seed, ne, el.Nq).numpy()
    return wl.point_values(seed, ne, el.Nq, ncomp=3).numpy()


def gpu_op(nk, op, basis, geom, lam, x, dev="cuda"):
    """Runs one operator through the binding; x numpy -> numpy result."""
    xt = torch.from_numpy(np.ascontiguousarray(x)).to(dev)
    ne = xt.shape[-2]
    nm, nq = basis.num_modes, basis.num_points

    def new(n):
        return torch.full((ne, n), float("nan"), dtype=torch.float64, device=dev)

    if op == "bwdtrans":
        y = new(nq)
        nk.bwdtrans(basis, xt, y)
    elif op == "iprod":
        y = new(nm)
        nk.iprod(basis, geom, xt, y)
    elif op == "physderiv":
        d = [new(nq) for _ in range(3)]
        nk.physderiv(basis, geom, xt, d[0], d[1], d[2])
        y = torch.stack(d)
    elif op == "iprod_deriv":
        y = new(nm)
        nk.iprod_deriv(basis, geom, xt[0].contiguous(), xt[1].contiguous(), xt[2].contiguous(), y)
    elif op == "mass":
        y = new(nm)
        nk.mass_apply(basis, geom, xt, y)
    elif op == "laplacian":
        y = new(nm)
        nk.laplacian_apply(basis, geom, xt, y)
    elif op == "helmholtz":
        y = new(nm)
        nk.helmholtz_apply(basis, geom, lam, xt, y)
    else:
        raise KeyError(op)
    torch.cuda.synchronize()
    return y.cpu().numpy()


def op_err(op, got, ref):
    if op == "physderiv":   # [3][ne][Nq]: judge the gradient as one vector per element
        return normwise_err(np.moveaxis(got, 0, 1), np.moveaxis(ref, 0, 1))
    return normwise_err(got, ref)
