"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

Holds no arithmetic of the method (see gen/fields.py).
"""
from .fields import (  # noqa: F401
    gauge_field, gauge_links, unit_gauge_field, spinor_field, site_parity,
    random_su3_per_site, reunitarise, gaussian, complex_gaussian,
)
