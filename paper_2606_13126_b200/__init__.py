"""MiniPIC hot path for B200 (sm_100a): paged attention over a position-free KV cache.

The product is the C-ABI library declared in ``include/minipic.h`` (built from
``paper_2606_13126_b200/csrc``).  This package holds

* ``binding``   - thin ctypes marshalling layer with the same call names,
* ``build``     - the in-tree nvcc build of ``libminipic.so``,
* ``workloads`` - seeded synthetic input generators (no method arithmetic).

Importing the package does not load the CUDA library; ``binding.lib()`` does and
fails loudly when it is missing.  Nothing here imports ``oracle/``.
"""

__all__ = ["binding", "build", "workloads"]
