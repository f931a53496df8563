"""B200-native channel-flow DNS substep + low-storage filter (arxiv 1808.06461).

The product is the C-ABI library ``libchan.so`` (paper_1808_06461_b200/csrc, include/chan.h) and the
thin ctypes binding in :mod:`paper_1808_06461_b200.binding`.  Importing the package does not load
the library; :func:`paper_1808_06461_b200.binding.load` does, and fails loudly if it is missing.
"""
