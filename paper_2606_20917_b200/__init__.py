"""paper_2606_20917_b200 -- Python face of libnk (include/nk.h): B200-native, matrix-free,
sum-factorised spectral/hp elemental operators (arxiv/paper_2606_20917 hot path).

The binding (binding.py) only marshals arguments; every step of the path runs in the CUDA
kernels of libnk.so.  Names are resolved lazily so that `python -m paper_2606_20917_b200.build`
can run before the library exists; any other use without a built libnk.so raises.
"""
_EXPORTS = ("lib", "NkError", "Basis", "Geom", "HEX", "TET", "PRISM", "bwdtrans", "iprod", "physderiv",
            "iprod_deriv", "mass_apply", "laplacian_apply", "helmholtz_apply", "helmholtz_apply_fields", "helmholtz_apply_blocks",
            "helmholtz_apply_host", "GatherScatter", "gs_gather", "gs_scatter_add", "assembled_helmholtz_apply", "assembled_helmholtz_apply_static", "static_max_local_dofs", "cg_solve", "Partition", "torch_allreduce", "part_exchange_sum", "part_assembled_helmholtz_apply", "part_cg_solve", "PRECOND_NONE", "PRECOND_JACOBI", "jit_compile_check", "jit_compile_check_kernel", "jit_stats", "set_affine_simplex_form", "get_affine_simplex_form", "probe_fp64_peak", "probe_fp64_dmma_peak", "launch_count", "version", "LIB_PATH", "DECLARED_SYMBOLS")


def __getattr__(name):
    if name in _EXPORTS:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)


__all__ = list(_EXPORTS)
