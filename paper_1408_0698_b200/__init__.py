"""B200-native Shack-Hartmann WFS hot path of arxiv/paper_1408_0698.

`paper_1408_0698_b200.binding` is the thin ctypes layer over the C-ABI library (include/shwfs.h);
`paper_1408_0698_b200.workloads` makes the seeded synthetic inputs.  Importing the package does not
load the CUDA library; the first call into `binding` does, and fails loudly if it is missing.
"""
__all__ = ["binding", "workloads", "build"]
