"""GPU parity at BASELINE.json's FULL sizes (configs 2, 3 and 5), in the launch configuration that
bench.py times (same generators, same calls), on sampled elements that the oracle computes one by one.
The sample always holds the first and last element, both ends of an interleave group, the ragged tail
of the last group and seeded random elements.  Gate: normwise 1e-12 (A18)."""
import numpy as np
import pytest
import torch

import nk_cases as K
from oracle import nk_oracle as o
from workloads import configs as cfgs
from workloads import synthetic as wl

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def nk():
    import paper_2606_20917_b200 as nk
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return nk


def sample_elements(ne, E, seed, nrand=48):
    fixed = [0, 1, E - 1, E, 2 * E - 1, ne // 2, ne - E - 1, ne - E, ne - 2, ne - 1]
    rng = np.random.Generator(np.random.Philox(seed))
    idx = sorted(set(int(i) for i in fixed if 0 <= i < ne) | set(int(i) for i in rng.integers(0, ne, nrand)))
    return torch.tensor(idx, dtype=torch.long)


def run_full(nk, cfg):
    dev = torch.device("cuda", 0)
    title, op, blocks = cfgs.config_blocks(cfg, device=dev)
    assert op == "helmholtz"
    work = []
    for b in blocks:
        basis = nk.Basis(b["shape"], b["P"])
        A, J = cfgs.block_factors(b, basis.points())
        geom = nk.Geom(basis, A, J, b["deformed"])
        ne = J.shape[0]
        x = wl.coefficients(b["seed"], ne, basis.num_modes).to(dev)
        y = torch.full_like(x, float("nan"))
        idx = sample_elements(ne, basis.interleave[int(b["deformed"])], b["seed"])
        As, Js = A[idx.to(dev)].cpu(), J[idx.to(dev)].cpu()
        del A, J
        work.append((b, basis, geom, x, y, idx, As, Js))
    lam = blocks[0]["lam"]
    if len(work) == 1:
        b, basis, geom, x, y = work[0][:5]
        nk.helmholtz_apply(basis, geom, lam, x, y)
    else:
        nk.helmholtz_apply_blocks([(w[1], w[2], w[3], w[4]) for w in work], lam)
    torch.cuda.synchronize()
    worst = 0.0
    for b, basis, geom, x, y, idx, As, Js in work:
        assert torch.isfinite(y).all(), "non-finite output in %s" % title
        el = K.element(b["shape"], b["P"])
        # the oracle evaluates the geometry of the sampled elements at ITS OWN quadrature points
        v0, E = b["v0"][idx.to(dev)].cpu(), b["E"][idx.to(dev)].cpu()
        Ao, Jo = (wl.sinusoidal_factors(v0, E, el.xi) if b["deformed"] else wl.affine_factors(v0, E))
        # the device evaluation of the generator (the kernel's input) and the host evaluation (the oracle's input) must
        # agree to rounding, or the parity gate below would measure the generator instead of the kernel
        assert np.abs(Ao.numpy() - As.numpy()).max() <= 1e-13 * np.abs(Ao.numpy()).max(), "input generator: device vs host"
        assert np.abs(Jo.numpy() - Js.numpy()).max() <= 1e-13 * np.abs(Jo.numpy()).max(), "input generator: device vs host"
        ref = o.helmholtz(el, Ao.numpy(), Jo.numpy(), b["lam"], x[idx.to(dev)].cpu().numpy())
        ys = y[idx.to(dev)].cpu().numpy()
        err = K.normwise_err(ys, ref)
        worst = max(worst, err)
        # shown by `pytest -s` (profiles/r2_repeat.md): how far the two evaluations of the input generator are apart
        print("%s shape %d: generator device vs host dA %.2e dJ %.2e; parity %.2e on %d sampled elements" % (
            title, b["shape"], np.abs(Ao.numpy() - As.numpy()).max() / np.abs(Ao.numpy()).max(),
            np.abs(Jo.numpy() - Js.numpy()).max() / np.abs(Jo.numpy()).max(), err, len(idx)))
        if err > TOL:   # say where: per-element errors and how far the two geometry evaluations are apart
            pe = np.abs(ys - ref).max(axis=1) / np.abs(ref).max(axis=1)
            where = [(int(idx[i]), "%.1e" % pe[i]) for i in np.argsort(-pe)[:6]]
            dA = np.abs(Ao.numpy() - As.numpy()).max() / np.abs(Ao.numpy()).max()
            dJ = np.abs(Jo.numpy() - Js.numpy()).max() / np.abs(Jo.numpy()).max()
            raise AssertionError("%s shape %d: normwise error %.3e on %d sampled elements; worst elements %s; "
                                 "geometry device vs host: dA %.2e dJ %.2e" % (title, b["shape"], err, len(idx), where, dA, dJ))
    return worst


def test_config2_full_size(nk):
    run_full(nk, 2)


def test_config3_full_size(nk):
    run_full(nk, 3)


def test_config5_full_size(nk):
    run_full(nk, 5)


@pytest.mark.parametrize("P", [1, 4, 7, 10])
def test_config4_full_size_sampled(nk, P):
    """config 4 (hex affine P-sweep, ~5e7 DoF): mass and Laplacian applied separately, sampled elements."""
    dev = torch.device("cuda", 0)
    title, op, blocks = cfgs.config_blocks(4, device=dev, P_sweep=P)
    b = blocks[0]
    basis = nk.Basis(b["shape"], P)
    A, J = cfgs.block_factors(b, basis.points())
    geom = nk.Geom(basis, A, J, False)
    ne = J.shape[0]
    x = wl.coefficients(b["seed"], ne, basis.num_modes).to(dev)
    ym, yl = torch.full_like(x, float("nan")), torch.full_like(x, float("nan"))
    nk.mass_apply(basis, geom, x, ym)
    nk.laplacian_apply(basis, geom, x, yl)
    torch.cuda.synchronize()
    idx = sample_elements(ne, basis.interleave[0], b["seed"], nrand=16 if P > 6 else 48).to(dev)
    el = K.element(o.HEX, P)
    An, Jn, xn = A[idx].cpu().numpy(), J[idx].cpu().numpy(), x[idx].cpu().numpy()
    assert K.normwise_err(ym[idx].cpu().numpy(), o.mass(el, Jn, xn)) <= TOL
    assert K.normwise_err(yl[idx].cpu().numpy(), o.laplacian(el, An, Jn, xn)) <= TOL


def _ones(basis, ne, dev):
    """coefficients of the constant function 1: the vertex modes (A8: they sum to 1)."""
    verts = {0: [(p, q, r) for p in (0, 1) for q in (0, 1) for r in (0, 1)],
             1: [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)],
             2: [(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0), (0, 0, 1), (0, 1, 1)]}[basis.shape]
    one = torch.zeros((ne, basis.num_modes), dtype=torch.float64, device=dev)
    for v in verts:
        m = basis.mode_index(*v)
        assert m >= 0
        one[:, m] = 1.0
    return one


@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_full_size_invariants_all_elements(nk, cfg):
    """Properties that hold at any size, checked on EVERY element of the BASELINE meshes (north_star
    invariants): integrating 1 gives the volume of the unit cube; the Laplacian annihilates constants;
    the Helmholtz operator is symmetric."""
    dev = torch.device("cuda", 0)
    title, op, blocks = cfgs.config_blocks(cfg, device=dev)
    vol = 0.0
    for b in blocks:
        basis = nk.Basis(b["shape"], b["P"])
        A, J = cfgs.block_factors(b, basis.points())
        geom = nk.Geom(basis, A, J, b["deformed"])
        ne = J.shape[0]
        del A, J
        one = _ones(basis, ne, dev)
        y = torch.empty_like(one)
        nk.mass_apply(basis, geom, one, y)
        vol += float((one * y).sum())
        x = wl.coefficients(b["seed"], ne, basis.num_modes).to(dev)
        z = wl.coefficients(b["seed"] + 1, ne, basis.num_modes).to(dev)
        lx = torch.empty_like(x)
        nk.laplacian_apply(basis, geom, x, lx)
        nk.laplacian_apply(basis, geom, one, y)
        scale = lx.abs().amax(dim=1)
        assert float((y.abs().amax(dim=1) / scale).max()) <= 1e-12, "L 1 != 0 (%s)" % title
        hx, hz = torch.empty_like(x), torch.empty_like(x)
        nk.helmholtz_apply(basis, geom, b["lam"], x, hx)
        nk.helmholtz_apply(basis, geom, b["lam"], z, hz)
        a1, a2 = (z * hx).sum(dim=1), (x * hz).sum(dim=1)           # per element: <z, H x> = <x, H z>
        den = (z.abs() * hx.abs()).sum(dim=1)
        assert float(((a1 - a2).abs() / den).max()) <= 1e-12, "H not symmetric (%s)" % title
    # config 5: the tets fill z in [0, 1/4) and the prisms the rest, together the unit cube
    tol = 1e-9 if blocks[0]["deformed"] else 1e-12     # the sinusoidal map integrates to 1 up to quadrature error
    assert abs(vol - 1.0) <= tol, "sum of element volumes %.15g (%s)" % (vol, title)


@pytest.mark.parametrize("cfg", [2, 3])
def test_full_size_every_element_against_the_oracle(nk, cfg):
    """configs 2 and 3 at BASELINE size, EVERY element against the oracle (oracle.parallel: the unchanged oracle
    over element chunks in a process pool on all host cores).  The oracle's inputs are evaluated on the host at
    the oracle's own quadrature points; the kernel's on the device at the library's."""
    from oracle.parallel import OraclePool
    dev = torch.device("cuda", 0)
    title, op, blocks = cfgs.config_blocks(cfg, device=dev)
    b = blocks[0]
    basis = nk.Basis(b["shape"], b["P"])
    A, J = cfgs.block_factors(b, basis.points())
    geom = nk.Geom(basis, A, J, b["deformed"], streams=nk.Geom.METRIC)
    ne = J.shape[0]
    del A, J
    x = wl.coefficients(b["seed"], ne, basis.num_modes)
    y = torch.full((ne, basis.num_modes), float("nan"), dtype=torch.float64, device=dev)
    nk.helmholtz_apply(basis, geom, b["lam"], x.to(dev), y)
    torch.cuda.synchronize()
    got = y.cpu().numpy()
    el = K.element(b["shape"], b["P"])
    v0, E = b["v0"].cpu(), b["E"].cpu()
    worst, step = 0.0, 8192
    with OraclePool() as pool:
        for s in range(0, ne, step):
            Ao, Jo = (wl.sinusoidal_factors(v0[s:s + step], E[s:s + step], el.xi) if b["deformed"]
                      else wl.affine_factors(v0[s:s + step], E[s:s + step]))
            ref = pool.apply("helmholtz", b["shape"], b["P"], b["P"] + 2, Ao.numpy(), Jo.numpy(), b["lam"], x[s:s + step].numpy())
            pe = np.abs(got[s:s + step] - ref).max(axis=1) / np.abs(ref).max(axis=1)
            worst = max(worst, float(pe.max()))
            assert pe.max() <= TOL, "%s: element %d normwise error %.3e" % (title, s + int(pe.argmax()), pe.max())
    print("%s: %d elements, worst normwise error %.2e" % (title, ne, worst))
