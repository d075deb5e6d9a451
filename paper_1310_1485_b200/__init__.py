"""B200-native ExB nonlinearity of GENE (arxiv 1310.1485, sect. 2): C-ABI library + thin binding.

`gene_nl_create / gene_nl_compute / gene_nl_destroy` (and the helpers of include/gene_nl.h) are
re-exported from `.binding`, which loads the in-tree CUDA shared library and FAILS LOUDLY if it is
missing -- there is no CPU fallback.  `.workloads` holds the seeded synthetic inputs.
"""
from . import workloads  # noqa: F401

_BINDING_NAMES = (
    "gene_nl_create", "gene_nl_compute", "gene_nl_compute_em", "gene_nl_destroy", "gene_nl_last_error", "GENE_NL_CHI_EM",
    "gene_nl_compute_host", "gene_nl_compute_em_host", "gene_nl_set_scratch_bytes", "gene_nl_set_plane_kernel", "GENE_NL_KERNEL_AUTO", "GENE_NL_KERNEL_CLUSTER", "GENE_NL_KERNEL_GROUP", "GENE_NL_KERNEL_BATCHED", "GENE_NL_KERNEL_WARP", "gene_nl_compute_profiled", "gene_nl_workspace_bytes", "gene_nl_launches_per_compute",
    "gene_nl_query", "gene_nl_compute_static", "gene_nl_probe_peaks", "GeneNL", "GeneNLError", "library_path", "load_library",
    "gene_nlx_create", "gene_nlx_compute", "gene_nlx_compute_host", "gene_nlx_destroy", "gene_nlx_query",
)


def __getattr__(name):
    if name in _BINDING_NAMES or name == "binding":
        import importlib
        mod = importlib.import_module(".binding", __name__)
        return mod if name == "binding" else getattr(mod, name)
    raise AttributeError(name)
