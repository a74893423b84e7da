"""B200-native D3Q19 LBM-LES stream-collide path of arxiv/paper_2607_04516.

``paper_2607_04516_b200.Lbm`` is the thin Python binding of the C-ABI library
(include/lbm.h).  Importing the package does not load the CUDA library; the
first use of the binding does, and fails loudly if it has not been built.
``paper_2607_04516_b200.workloads`` holds the seeded synthetic inputs.
"""


def __getattr__(name):
    if name in ("Lbm", "load_library", "library_path", "LbmError"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
