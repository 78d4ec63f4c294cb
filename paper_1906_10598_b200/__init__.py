"""B200-native phase tracking by Differential Evolution (arxiv 1906.10598, hot path only).

``paper_1906_10598_b200.pt``         thin ctypes binding of the C-ABI library ``libpt.so`` (CUDA, sm_100a)
``paper_1906_10598_b200.workloads``  seeded synthetic inputs (numpy only; shared with the tests' oracle side)
``paper_1906_10598_b200.build``      nvcc build of ``libpt.so`` (in-tree)
``paper_1906_10598_b200.shard``      one track over several GPUs: block ranges per rank + one all-gather (torch.distributed)

Importing the package loads nothing; the CUDA library is loaded on the first call into ``pt`` and
there is no CPU fallback: a missing or unloadable ``libpt.so`` raises.
"""
__all__ = ["pt", "workloads", "build", "shard"]
