"""B200-native thermal two-component D2Q9 lattice-Boltzmann step (TLBfind, arXiv 2109.12565).

The CUDA binding loads the C-ABI shared library on first use and fails loudly if it is missing -- there is no
CPU fallback.  The package holds the product only: the seeded input generators that feed both it and the oracle in the
tests live in the top-level `inputs` module.
"""


def __getattr__(name):
    if name in ("TLB", "binding", "load_library", "TLBError", "default_params"):
        import importlib
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    raise AttributeError(name)
