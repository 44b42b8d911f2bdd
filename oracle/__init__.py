"""CPU oracle of the realfast search hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU-baseline /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1802_03084_b200`` (the CUDA path) and imports nothing from it.
"""
from .realfast_oracle import (  # noqa: F401
    K_DM,
    C_LIGHT,
    Candidate,
    mean_subtract,
    candidate_spectrum,
    inject_transient,
    periodicity_nt,
    periodicity_spectrum,
    periodicity_image,
    periodicity_stats,
    periodicity_search,
    delay_table,
    cell_table,
    dedisperse_resample,
    grid_visibilities,
    image_from_grid,
    image_direct_dft,
    image_stats,
    n_images,
    search,
    search_image,
)
