"""B200-native mixed-step absorbed-MLA attention for deflected prefills (KAIROS, arxiv 2607.02043).

`paper_2607_02043_b200.kairos`   -- thin ctypes binding over the C-ABI library (libkairos.so, CUDA sm_100a);
                                    importing it fails loudly if the library is not built.
`paper_2607_02043_b200.workloads` -- seeded synthetic input generators (numpy only, no attention arithmetic).
`paper_2607_02043_b200.build`     -- nvcc build of csrc/ -> libkairos.so (in-tree).
"""
from . import workloads  # noqa: F401

__all__ = ["workloads"]
