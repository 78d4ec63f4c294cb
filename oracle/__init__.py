"""fp64 CPU oracle of the phase-tracking hot path (arxiv 1906.10598).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  It imports
nothing from ``paper_1906_10598_b200`` and shares no code with the CUDA path.

``oracle/pt_oracle.c`` holds the arithmetic (plain C, fp64, exact-integer Philox); this package
only compiles it with gcc and marshals numpy arrays into it with ctypes.  ``oracle/pt_acquire.py`` is the
fp64 numpy statement of the paper's initial range determination (FFT acquisition).
"""
from .pt_acquire import acquire, piece_estimate  # noqa: F401
from .pt_retry import doubtful_blocks, extrapolated_box, refit_doubtful  # noqa: F401
from .pt_oracle import (  # noqa: F401
    aux_uniforms,
    build,
    cor,
    cr32,
    de_trial,
    de_draws,
    default_t0,
    doppler_products,
    fcor_of_cor,
    fit_blocks,
    fitness,
    indices_from_words,
    init_uniforms,
    model,
    num_threads,
    philox4x32_10,
    rss,
    unpack_samples,
)
