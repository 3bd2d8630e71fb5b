"""B200-native per-timestep update of the Microcosmos world (arxiv/paper_2607_02954).

`worlds` holds the seeded input generators; `binding` is the thin ctypes layer over the
C-ABI library (include/mc.h) whose kernels do every step of the path.  There is no CPU
fallback: using `binding` without the built CUDA library raises.
"""
