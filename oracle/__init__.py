"""CPU oracle for the mixed-variational plane-wave band-structure path (arXiv:1310.6380).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_1310_6380_b200/`` may import this
package; only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` do.  It shares no code with the CUDA path.
"""
from .bandstructure import (  # noqa: F401
    reciprocal_basis,
    plane_wave_indices,
    shape_integral,
    polygon_area,
    polygon_centroid,
    shape_integral_centroid,
    isotropic_plane_strain_compliance,
    lame_from_C11_C44,
    voigt_compliance,
    assemble_direct,
    shape_integral_table,
    assemble,
    coupling_B,
    pencil_K,
    bands_at_k,
    modes_at_k,
    band_structure,
    omega_svd_route,
)
