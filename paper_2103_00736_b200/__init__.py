"""B200-native hot path of arXiv 2103.00736 (operator-splitting conic solver + adaptive conditioning).

The package holds three things only:

* ``csrc/``      -- the CUDA kernels and the C-ABI library ``libcs.so`` (``include/cs.h``);
* ``binding``    -- a thin ctypes binding with the same ``cs_*`` names (argument marshalling only);
* ``workloads``  -- the seeded synthetic input generators (no solver arithmetic), shared with the tests'
                    oracle side.

Nothing is imported eagerly: ``workloads`` must stay importable without the CUDA library, and the
binding must fail loudly (not fall back) when ``libcs.so`` is missing.
"""

__all__ = ["binding", "workloads", "build"]
