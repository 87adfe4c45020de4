"""B200-native per-cell two-temperature radiative cooling step of arXiv 2505.08855.

The public calls mirror the C ABI of ``include/cool.h`` (``cool_table_build_host``,
``cool_table_create``, ``cool_apply``, ``cool_table_destroy``) and live in ``.api``; they
only marshal arguments — every step of the path runs in the CUDA kernels of ``csrc/``.
Importing the package is cheap; the shared library is loaded on first use and the import
fails loudly if it is missing.  ``.synth`` (seeded inputs) is numpy-only.
"""
__all__ = ["api", "synth"]
