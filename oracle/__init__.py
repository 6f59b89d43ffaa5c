"""CPU oracle for the SSFM hot path of arxiv/paper_2410_04994 -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs of
``bench.py`` may import this package.  It shares no code with ``paper_2410_04994_b200`` (the CUDA path)
and never imports it.  See ``shg_oracle.h`` for what is pinned and what is "parity unpinned".
"""
from .oracle import (  # noqa: F401
    Oracle,
    build,
    dft2_brute,
    fft2,
    gaussian_input,
    num_threads,
    set_num_threads,
)
