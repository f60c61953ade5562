"""B200-native gint_vlocal: real-space grid integration of the local-potential
Hamiltonian in NAO-based RT-TDDFT (Sec. 3.3.1, Eq. 45).

    from paper_2603_21835_b200 import gint_setup
    ctx = gint_setup(lattice, ngrid, species, atom_species, atom_pos)
    H = ctx.gint_vlocal(V_dev)            # CUDA float64 tensors
    iat, jat, R, offset = ctx.gint_get_blocks()

`workloads` (seeded synthetic inputs) imports without the CUDA library; the
binding does not: there is no CPU fallback.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    if name in ("gint_setup", "gint_measure_fp64_peak", "gint_fold_k_static_max_blocks", "GintContext", "GintError", "binding"):
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)
