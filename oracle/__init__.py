"""CPU oracle for the biobeam split-step BPM hot path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1706_02261_b200`` (the CUDA path) and never imports it.

The arithmetic lives in ``bpm_oracle.c`` (plain C, IEEE double, its own
radix-2 FFT); this module only marshals numpy arrays through ctypes.
See ``bpm_oracle.c``'s header for what it follows in the paper and how it is
pinned.
"""
from .bpm_oracle import (  # noqa: F401
    build,
    dft2_bruteforce,
    fft1,
    fft2,
    bpm_step,
    bpm_step_backward,
    propagate,
    propagate_stream,
    multiplex_psf,
    nref_from_dn,
    num_threads,
    propagate_backward,
    refocus,
    extract_tiles,
    lightsheet,
    multiplex_annular,
    image_formation,
)
