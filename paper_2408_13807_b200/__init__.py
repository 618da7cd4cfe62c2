"""dies-b200: the data-parallel hot path of DIES (arXiv 2408.13807) as hand-written sm_100a CUDA.

`paper_2408_13807_b200.binding` wraps the C ABI of include/dies.h (argument marshalling only);
`paper_2408_13807_b200.synth` generates the seeded synthetic inputs.  Nothing here computes any step of the
method on the CPU: without the CUDA library and a B200 every call fails loudly.
"""
__all__ = ["binding", "synth", "build"]
