"""B200-native attention hot path of PrefixFlow's training-time KV cache (arxiv/paper_2606_01143).

Public surface = the Python binding of the C-ABI library (`include/prefixflow.h`):
`pf_create`, `pf_group_begin`, `pf_phaseA_fwd`, `pf_phaseB_fwd`, `pf_phaseB_bwd`,
`pf_phaseC_bwd`, `pf_group_end`, ... re-exported from `binding`. Every step of the path runs in
the CUDA kernels under `csrc/`; PyTorch is used for device memory and streams only.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs"]
