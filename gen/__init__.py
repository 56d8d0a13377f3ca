"""Seeded synthetic-input generators shared by the oracle tests and the CUDA harness.

This package holds NO arithmetic of the method (no orbitals, no densities, no MLP):
only geometry recipes, random weights and the byte layout of the weights blob
(SURVEY.md section 8(b), 8(d)). Both `oracle/` and `paper_2505_06711_b200/` parse
the blob with their own code.
"""
from .configs import CONFIGS, make_config, water_box, fcc_lattice, maxwell_boltzmann  # noqa: F401
from .weights import make_weights, pack_blob, blob_layout, n_orb_default, n_monomials  # noqa: F401
