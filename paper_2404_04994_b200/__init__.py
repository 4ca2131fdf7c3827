"""B200-native ground-state charge search of the constant capacitance model (arXiv 2404.04994, "QArray").

The product is the C-ABI library ``libqarray_b200.so`` (include/qarray_b200.h; sources in ``csrc/``).  ``api`` is the
thin Python binding over it (argument marshalling only); ``workloads`` builds the seeded synthetic inputs.  Importing
this package does not load the library; ``paper_2404_04994_b200.api`` does, and fails loudly if it is missing.
"""
__all__ = ["api", "workloads", "build"]
