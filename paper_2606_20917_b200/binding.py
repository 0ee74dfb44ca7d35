"""ctypes binding of libnk.so -- same names as include/nk.h, argument marshalling only.

PyTorch is used for device memory and streams; tensors are passed as raw pointers.  There is no
Python or CPU implementation behind these calls: if libnk.so is missing the import fails.
"""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NK_LIB") or os.path.join(HERE, "libnk.so")   # NK_LIB: another build of the same library
HEX, TET, PRISM = 0, 1, 2
TAB_NODES, TAB_WEIGHTS, TAB_DERIV, TAB_PSI, TAB_KRON = 0, 1, 2, 3, 4

if not os.path.exists(LIB_PATH):
    raise ImportError("libnk.so not built (%s): run `python -m paper_2606_20917_b200.build`; "
                      "there is no CPU fallback" % LIB_PATH)
lib = C.CDLL(LIB_PATH)

_p, _d, _i, _i64, _sz = C.c_void_p, C.c_double, C.c_int, C.c_int64, C.c_size_t
_SIG = {
    "nk_basis_create": (_i, [_i, _i, _i, C.POINTER(_p)]),
    "nk_basis_destroy": (_i, [_p]),
    "nk_basis_num_modes": (_i, [_p]),
    "nk_basis_num_points": (_i, [_p]),
    "nk_basis_interleave": (_i, [_p, _i]),
    "nk_basis_get_table": (_i, [_p, _i, _i, C.POINTER(_d), _sz, C.POINTER(_sz)]),
    "nk_basis_mode_index": (_i, [_p, _i, _i, _i]),
    "nk_basis_get_points": (_i, [_p, C.POINTER(_d), _sz]),
    "nk_geom_upload": (_i, [_p, _i64, _i, _p, _p, _i, _p, C.POINTER(_p)]),
    "nk_geom_upload_streams": (_i, [_p, _i64, _i, _p, _p, _i, C.c_uint, _p, C.POINTER(_p)]),
    "nk_geom_destroy": (_i, [_p]),
    "nk_geom_num_elements": (_i64, [_p]),
    "nk_bwdtrans": (_i, [_p, _i64, _p, _p, _p]),
    "nk_iprod": (_i, [_p, _p, _p, _p, _p]),
    "nk_physderiv": (_i, [_p, _p, _p, _p, _p, _p, _p]),
    "nk_iprod_deriv": (_i, [_p, _p, _p, _p, _p, _p, _p]),
    "nk_mass_apply": (_i, [_p, _p, _p, _p, _p]),
    "nk_laplacian_apply": (_i, [_p, _p, _p, _p, _p]),
    "nk_helmholtz_apply": (_i, [_p, _p, _d, _p, _p, _p]),
    "nk_helmholtz_apply_fields": (_i, [_p, _p, _d, _i, C.POINTER(_p), C.POINTER(_p), _p]),
    "nk_helmholtz_apply_blocks": (_i, [_i, _p, _d, _p]),
    "nk_helmholtz_apply_host": (_i, [_p, _p, _d, _p, _p, _p]),
    "nk_gs_create": (_i, [_i64, _i, _i64, _p, _p, C.POINTER(_p)]),
    "nk_gs_destroy": (_i, [_p]),
    "nk_gs_num_global": (_i64, [_p]),
    "nk_gs_set_constrained": (_i, [_p, _i64, _p]),
    "nk_gs_gather": (_i, [_p, _p, _p, _p]),
    "nk_gs_scatter_add": (_i, [_p, _p, _p, _p]),
    "nk_assembled_helmholtz_apply": (_i, [_p, _p, _p, _d, _p, _p, _p]),
    "nk_static_max_local_dofs": (_i64, []),
    "nk_assembled_helmholtz_apply_static": (_i, [_p, _p, _p, _d, _p, _p, _p]),
    "nk_cg_solve": (_i, [_p, _p, _p, _d, _p, _p, _i, _d, _i, C.POINTER(_i), C.POINTER(_d), _p]),
    "nk_part_create": (_i, [_p, _i64, _p, _p, _p, _i64, _p, _p, C.POINTER(_p)]),
    "nk_part_destroy": (_i, [_p]),
    "nk_part_exchange_sum": (_i, [_p, _p, _p]),
    "nk_part_assembled_helmholtz_apply": (_i, [_p, _p, _p, _d, _p, _p, _p]),
    "nk_part_cg_solve": (_i, [_p, _p, _p, _d, _p, _p, _i, _d, _i, C.POINTER(_i), C.POINTER(_d), _p]),
    "nk_jit_compile_check": (_i, [_i, C.POINTER(_d), C.POINTER(_sz)]),
    "nk_jit_compile_check_kernel": (_i, [_i, _i, _i, _i, _i, C.POINTER(_d), C.POINTER(_sz)]),
    "nk_jit_stats": (_i, [C.POINTER(_i64), C.POINTER(_d)]),
    "nk_set_affine_simplex_form": (_i, [_i]),
    "nk_get_affine_simplex_form": (_i, []),
    "nk_basis_get_reference_matrix": (_i, [_p, _i, C.POINTER(_d), _sz]),
    "nk_probe_fp64_peak": (_i, [_i, C.POINTER(_d), C.POINTER(_d)]),
    "nk_probe_fp64_dmma_peak": (_i, [_i, C.POINTER(_d), C.POINTER(_d)]),
    "nk_launch_count": (_i64, []),
    "nk_last_error": (C.c_char_p, []),
    "nk_version": (C.c_char_p, []),
}
DECLARED_SYMBOLS = tuple(_SIG)
for _name, (_res, _args) in _SIG.items():
    _f = getattr(lib, _name)          # AttributeError here = the .so does not export what nk.h declares
    _f.restype, _f.argtypes = _res, _args


class NkBlock(C.Structure):
    _fields_ = [("basis", _p), ("geom", _p), ("inp", _p), ("out", _p)]


class NkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("nk_status %d: %s" % (code, msg))
        self.code = code


def _check(code):
    if code != 0:
        raise NkError(code, lib.nk_last_error().decode())


def _ptr(t, allow_none=False):
    if t is None:
        if allow_none:
            return None
        raise ValueError("tensor required")
    if t.dtype != torch.float64 or not t.is_contiguous():
        raise ValueError("libnk takes contiguous float64 tensors")
    return t.data_ptr()


def _dev_ptr(t, allow_none=False):
    if t is not None and not t.is_cuda:
        raise ValueError("device tensor required (libnk has no CPU path)")
    return _ptr(t, allow_none)


# torch.cuda.current_stream() costs 3 us per call, as much as a small kernel: take the raw handle of torch's
# current stream directly when this torch has the private accessors (same stream, 0.3 us)
_raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)
_raw_device = getattr(torch._C, "_cuda_getDevice", None)


def _stream(stream=None):
    if stream is not None:
        return stream.cuda_stream
    if _raw_stream is not None and _raw_device is not None:
        return _raw_stream(_raw_device())
    return torch.cuda.current_stream().cuda_stream


class Basis:
    """nk_basis handle (host precompute only; needs no GPU)."""

    def __init__(self, shape, P, Q=None):
        Q = P + 2 if Q is None else Q
        h = _p()
        _check(lib.nk_basis_create(shape, P, Q, C.byref(h)))
        self.h, self.shape, self.P, self.Q = h, shape, P, Q
        self.num_modes = lib.nk_basis_num_modes(h)
        self.num_points = lib.nk_basis_num_points(h)
        self.interleave = (lib.nk_basis_interleave(h, 0), lib.nk_basis_interleave(h, 1))   # (affine, deformed)

    def table(self, which, direction):
        n = _sz()
        _check(lib.nk_basis_get_table(self.h, which, direction, None, 0, C.byref(n)))
        buf = (_d * n.value)()
        _check(lib.nk_basis_get_table(self.h, which, direction, buf, n.value, None))
        return torch.tensor(list(buf), dtype=torch.float64)

    def points(self):
        """xi [Nq][3] of the quadrature points (input to geometry generators)."""
        buf = (_d * (3 * self.num_points))()
        _check(lib.nk_basis_get_points(self.h, buf, 3 * self.num_points))
        return torch.tensor(list(buf), dtype=torch.float64).reshape(self.num_points, 3)

    def mode_index(self, p, q, r):
        return lib.nk_basis_mode_index(self.h, p, q, r)

    def reference_matrix(self, c):
        """matrix c = 0..6 of the standard element [Nm][Nm] (nk_basis_get_reference_matrix; host only)."""
        n = self.num_modes * self.num_modes
        buf = (_d * n)()
        _check(lib.nk_basis_get_reference_matrix(self.h, c, buf, n))
        return torch.frombuffer(buf, dtype=torch.float64).clone().reshape(self.num_modes, self.num_modes)

    def close(self):
        if self.h:
            lib.nk_basis_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Geom:
    """nk_geom handle.  dxi_dx [nelem][npt][3][3], detJ [nelem][npt]; host or device tensors."""

    METRIC, FACTORS = 1, 2

    def __init__(self, basis, dxi_dx, detJ, deformed, stream=None, streams=3):
        nelem = detJ.shape[0]
        npt = basis.num_points if deformed else 1
        if tuple(dxi_dx.shape) != (nelem, npt, 3, 3) or tuple(detJ.shape) != (nelem, npt):
            raise ValueError("geometry shapes must be [nelem][%d][3][3] and [nelem][%d]" % (npt, npt))
        if dxi_dx.is_cuda != detJ.is_cuda:
            raise ValueError("dxi_dx and detJ must live on the same side")
        h = _p()
        _check(lib.nk_geom_upload_streams(basis.h, nelem, int(bool(deformed)), _ptr(dxi_dx), _ptr(detJ),
                                          int(dxi_dx.is_cuda), int(streams), _stream(stream), C.byref(h)))
        self.h, self.basis, self.nelem, self.deformed = h, basis, nelem, bool(deformed)

    def close(self):
        if self.h:
            lib.nk_geom_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _field(t, n, what, allow_none=False):
    """device pointer of a field tensor after checking its size (the C-ABI takes no sizes for field buffers: a
    short tensor would be a silent out-of-bounds device access) and its device.  Marshalling only."""
    if t is None:
        if allow_none:
            return None
        raise ValueError("%s: tensor required" % what)
    if t.numel() != n:
        raise ValueError("%s holds %d values, the block needs %d" % (what, t.numel(), n))
    if t.is_cuda and t.device.index != torch.cuda.current_device():
        raise ValueError("%s lives on cuda:%d, the current device is cuda:%d" % (what, t.device.index, torch.cuda.current_device()))
    return _dev_ptr(t)


def _no_alias(ins, outs):
    """nk.h: in/out must not alias (checked for every pair here; the library checks the first pair only)."""
    a = [t.data_ptr() for t in ins if t is not None]
    b = [t.data_ptr() for t in outs if t is not None]
    if set(a) & set(b) or len(set(b)) != len(b):
        raise ValueError("input and output tensors must be distinct buffers")


def bwdtrans(basis, coeffs, phys, stream=None):
    ne = coeffs.shape[0]
    _no_alias([coeffs], [phys])
    _check(lib.nk_bwdtrans(basis.h, ne, _field(coeffs, ne * basis.num_modes, "coeffs"),
                           _field(phys, ne * basis.num_points, "phys"), _stream(stream)))


def iprod(basis, geom, phys, coeffs, stream=None):
    _no_alias([phys], [coeffs])
    _check(lib.nk_iprod(basis.h, geom.h, _field(phys, geom.nelem * basis.num_points, "phys"),
                        _field(coeffs, geom.nelem * basis.num_modes, "coeffs"), _stream(stream)))


def physderiv(basis, geom, phys, d0, d1, d2, stream=None):
    nq = geom.nelem * basis.num_points
    _no_alias([phys], [d0, d1, d2])
    _check(lib.nk_physderiv(basis.h, geom.h, _field(phys, nq, "phys"), _field(d0, nq, "d0", True), _field(d1, nq, "d1", True),
                            _field(d2, nq, "d2", True), _stream(stream)))


def iprod_deriv(basis, geom, g0, g1, g2, coeffs, stream=None):
    nq = geom.nelem * basis.num_points
    _no_alias([g0, g1, g2], [coeffs])
    _check(lib.nk_iprod_deriv(basis.h, geom.h, _field(g0, nq, "g0", True), _field(g1, nq, "g1", True), _field(g2, nq, "g2", True),
                              _field(coeffs, geom.nelem * basis.num_modes, "coeffs"), _stream(stream)))


def _coeff_pair(basis, geom, inp, out):
    n = geom.nelem * geom.basis.num_modes     # sized by the geometry's own basis; a mismatching `basis` is the library's to refuse
    return _field(inp, n, "in"), _field(out, n, "out")


def mass_apply(basis, geom, inp, out, stream=None):
    pi, po = _coeff_pair(basis, geom, inp, out)
    _check(lib.nk_mass_apply(basis.h, geom.h, pi, po, _stream(stream)))


def laplacian_apply(basis, geom, inp, out, stream=None):
    pi, po = _coeff_pair(basis, geom, inp, out)
    _check(lib.nk_laplacian_apply(basis.h, geom.h, pi, po, _stream(stream)))


def helmholtz_apply(basis, geom, lam, inp, out, stream=None):
    pi, po = _coeff_pair(basis, geom, inp, out)
    _check(lib.nk_helmholtz_apply(basis.h, geom.h, float(lam), pi, po, _stream(stream)))


def helmholtz_apply_fields(basis, geom, lam, inps, outs, stream=None):
    """inps / outs: sequences of nfields device tensors [nelem][Nm] sharing the geometry of `geom`."""
    n = len(inps)
    if n != len(outs):
        raise ValueError("as many outputs as inputs")
    nn = geom.nelem * basis.num_modes
    pin = (_p * n)(*[_field(t, nn, "in[%d]" % k) for k, t in enumerate(inps)])
    pout = (_p * n)(*[_field(t, nn, "out[%d]" % k) for k, t in enumerate(outs)])
    _check(lib.nk_helmholtz_apply_fields(basis.h, geom.h, float(lam), n, pin, pout, _stream(stream)))


def helmholtz_apply_blocks(blocks, lam, stream=None):
    """blocks: sequence of (basis, geom, inp, out)."""
    arr = (NkBlock * len(blocks))()
    for k, (b, g, x, y) in enumerate(blocks):
        pi, po = _coeff_pair(b, g, x, y)
        arr[k] = NkBlock(b.h, g.h, pi, po)
    _check(lib.nk_helmholtz_apply_blocks(len(blocks), arr, float(lam), _stream(stream)))


def helmholtz_apply_host(basis, geom, lam, host_in, host_out, stream=None):
    if host_in.is_cuda or host_out.is_cuda:
        raise ValueError("host tensors required")
    n = geom.nelem * basis.num_modes
    if host_in.numel() != n or host_out.numel() != n:
        raise ValueError("host buffers must hold nelem x Nm = %d values" % n)
    _check(lib.nk_helmholtz_apply_host(basis.h, geom.h, float(lam), _ptr(host_in), _ptr(host_out), _stream(stream)))


class GatherScatter:
    """nk_gs handle.  l2g: int64 CPU tensor [nelem][Nm]; sign: int8 CPU tensor of +-1 or None."""

    def __init__(self, l2g, nglobal, sign=None):
        if l2g.dtype != torch.int64 or l2g.is_cuda or not l2g.is_contiguous() or l2g.dim() != 2:
            raise ValueError("l2g: contiguous int64 host tensor [nelem][Nm]")
        if sign is not None and (sign.dtype != torch.int8 or sign.is_cuda or not sign.is_contiguous() or sign.shape != l2g.shape):
            raise ValueError("sign: contiguous int8 host tensor of the shape of l2g")
        h = _p()
        _check(lib.nk_gs_create(l2g.shape[0], l2g.shape[1], int(nglobal), l2g.data_ptr(), sign.data_ptr() if sign is not None else None,
                                C.byref(h)))
        self.h, self.nelem, self.nm, self.nglobal = h, l2g.shape[0], l2g.shape[1], int(nglobal)

    def set_constrained(self, dofs):
        """dofs: int64 CPU tensor of constrained (Dirichlet) global dofs; empty removes the constraints."""
        if dofs.dtype != torch.int64 or dofs.is_cuda or not dofs.is_contiguous():
            raise ValueError("dofs: contiguous int64 host tensor")
        _check(lib.nk_gs_set_constrained(self.h, dofs.numel(), dofs.data_ptr() if dofs.numel() else None))

    def close(self):
        if self.h:
            lib.nk_gs_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def gs_gather(gs, glob, local, stream=None):
    _check(lib.nk_gs_gather(gs.h, _field(glob, gs.nglobal, "global"), _field(local, gs.nelem * gs.nm, "local"), _stream(stream)))


def gs_scatter_add(gs, local, glob, stream=None):
    _check(lib.nk_gs_scatter_add(gs.h, _field(local, gs.nelem * gs.nm, "local"), _field(glob, gs.nglobal, "global"), _stream(stream)))


def assembled_helmholtz_apply(basis, geom, gs, lam, inp, out, stream=None):
    _check(lib.nk_assembled_helmholtz_apply(basis.h, geom.h, gs.h, float(lam), _field(inp, gs.nglobal, "in"),
                                            _field(out, gs.nglobal, "out"), _stream(stream)))


def static_max_local_dofs():
    return int(lib.nk_static_max_local_dofs())


def assembled_helmholtz_apply_static(basis, geom, gs, lam, inp, out, stream=None):
    """nk_assembled_helmholtz_apply_static: the same operation with the work space in the library's static device array
    (allocates nothing; at most static_max_local_dofs() local dofs; calls that overlap on the GPU race on the array)."""
    _check(lib.nk_assembled_helmholtz_apply_static(basis.h, geom.h, gs.h, float(lam), _field(inp, gs.nglobal, "in"),
                                                   _field(out, gs.nglobal, "out"), _stream(stream)))


PRECOND_NONE, PRECOND_JACOBI = 0, 1


def cg_solve(basis, geom, gs, lam, rhs, x, rtol=1e-10, maxit=1000, precond=PRECOND_JACOBI, stream=None):
    """returns (iterations, relative residual); x holds the initial guess on entry and the solution on return."""
    it, rel = _i(), _d()
    _check(lib.nk_cg_solve(basis.h, geom.h, gs.h, float(lam), _field(rhs, gs.nglobal, "rhs"), _field(x, gs.nglobal, "x"),
                           int(precond), float(rtol), int(maxit), C.byref(it), C.byref(rel), _stream(stream)))
    return it.value, rel.value


# ---- the assembled system on a mesh split over ranks (include/nk.h: nk_part_*) ----
_ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)


class _DevicePtr:
    """a device pointer of n doubles as seen by torch.as_tensor (no copy)"""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f8", "data": (int(ptr), False), "version": 2}


def torch_allreduce(group=None):
    """the all-reduce of a Partition over torch.distributed (NCCL over NVLink on GPUs): sums the tensor in place"""
    import torch.distributed as dist

    def f(t):
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return f


class Partition:
    """nk_part handle: this rank's share of a mesh split over ranks.  shared_dof / shared_slot: int64 CPU tensors,
    shared_mult: int32 CPU tensor (workloads.assembly.partition_l2g produces them); allreduce(tensor): sums a float64 CUDA
    tensor in place over all ranks on the current stream (torch_allreduce(), or any callable for tests)."""

    def __init__(self, gs, shared_dof, shared_slot, shared_mult, n_interface, allreduce):
        for t, dt in ((shared_dof, torch.int64), (shared_slot, torch.int64), (shared_mult, torch.int32)):
            if t.dtype != dt or t.is_cuda or not t.is_contiguous() or t.numel() != shared_dof.numel():
                raise ValueError("shared_dof / shared_slot: contiguous int64 host tensors, shared_mult: int32, of one length")

        def cb(user, buf, n, stream):
            try:
                allreduce(torch.as_tensor(_DevicePtr(buf, n), device="cuda"))
                return 0
            except Exception:          # never let an exception cross the C boundary
                import traceback
                traceback.print_exc()
                return 1
        self._cb = _ALLREDUCE_FN(cb)   # kept alive as long as the handle
        ns = shared_dof.numel()
        h = _p()
        _check(lib.nk_part_create(gs.h, ns, shared_dof.data_ptr() if ns else None, shared_slot.data_ptr() if ns else None,
                                  shared_mult.data_ptr() if ns else None, int(n_interface), C.cast(self._cb, _p), None, C.byref(h)))
        self.h, self.gs = h, gs

    def close(self):
        if self.h:
            lib.nk_part_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def part_exchange_sum(part, vec, stream=None):
    _check(lib.nk_part_exchange_sum(part.h, _field(vec, part.gs.nglobal, "vec"), _stream(stream)))


def part_assembled_helmholtz_apply(basis, geom, part, lam, inp, out, stream=None):
    gs = part.gs
    _check(lib.nk_part_assembled_helmholtz_apply(basis.h, geom.h, part.h, float(lam), _field(inp, gs.nglobal, "in"),
                                                 _field(out, gs.nglobal, "out"), _stream(stream)))


def part_cg_solve(basis, geom, part, lam, rhs, x, rtol=1e-10, maxit=1000, precond=PRECOND_JACOBI, stream=None):
    """nk_part_cg_solve: (iterations, relative residual), identical on every rank; collective."""
    gs = part.gs
    it, rel = _i(), _d()
    _check(lib.nk_part_cg_solve(basis.h, geom.h, part.h, float(lam), _field(rhs, gs.nglobal, "rhs"), _field(x, gs.nglobal, "x"),
                                int(precond), float(rtol), int(maxit), C.byref(it), C.byref(rel), _stream(stream)))
    return it.value, rel.value


def jit_compile_check(nmodes):
    """(compile ms, cubin bytes) of the NVRTC specialisation of the reference-matrix Helmholtz kernel; needs no GPU."""
    ms, nb = _d(), _sz()
    _check(lib.nk_jit_compile_check(int(nmodes), C.byref(ms), C.byref(nb)))
    return ms.value, nb.value


def jit_compile_check_kernel(shape, P, Q, deformed, op):
    """NVRTC-compiles one sum-factorised instantiation without loading it (no GPU needed): (ms, cubin bytes)."""
    ms, nb = _d(), _sz()
    _check(lib.nk_jit_compile_check_kernel(int(shape), int(P), int(Q), int(bool(deformed)), int(op), C.byref(ms), C.byref(nb)))
    return ms.value, nb.value


def jit_stats():
    """(kernels specialised at run time for launching so far, their total NVRTC time in ms)"""
    k, ms = _i64(), _d()
    _check(lib.nk_jit_stats(C.byref(k), C.byref(ms)))
    return k.value, ms.value


def set_affine_simplex_form(form):
    """0 = automatic, 1 = sum-factorised, 2 = reference-matrix (nk_set_affine_simplex_form)."""
    _check(lib.nk_set_affine_simplex_form(int(form)))


def get_affine_simplex_form():
    return lib.nk_get_affine_simplex_form()


def probe_fp64_peak(iters=200):
    tf, ms = _d(), _d()
    _check(lib.nk_probe_fp64_peak(iters, C.byref(tf), C.byref(ms)))
    return tf.value, ms.value


def probe_fp64_dmma_peak(iters=200):
    tf, ms = _d(), _d()
    _check(lib.nk_probe_fp64_dmma_peak(iters, C.byref(tf), C.byref(ms)))
    return tf.value, ms.value


def launch_count():
    return lib.nk_launch_count()


def version():
    return lib.nk_version().decode()
