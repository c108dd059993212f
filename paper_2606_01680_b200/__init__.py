"""optcc-b200: B200-native execution of OPTCC AllReduce schedules (arxiv/paper_2606_01680).

`paper_2606_01680_b200.binding` is the thin ctypes layer over the C-ABI library (liboptcc.so);
`paper_2606_01680_b200.workloads` holds the seeded synthetic inputs.  Importing the package loads nothing.
"""
__all__ = ["binding", "workloads"]
