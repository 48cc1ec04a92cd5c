"""osdp-b200: operator-split transformer MLP (OSDP, arxiv 2305.09940 §3.3) for one B200.

The package holds only what the hot path needs:

* ``csrc/``     hand-written sm_100a CUDA kernels + the C-ABI (``include/osdp.h``)
* ``binding``   thin ctypes binding with the same names as the C-ABI (argument marshalling only)
* ``inputs``    seeded synthetic input generators (no arithmetic of the method)
* ``build``     the nvcc command that produces ``libosdp_b200.so`` in-tree

Nothing here imports ``oracle/``; the oracle is test infrastructure.
Sub-modules are imported lazily so that ``import paper_2305_09940_b200.inputs`` does not load
the CUDA library.
"""

__all__ = ["binding", "inputs", "build"]
__version__ = "0.1.0"
