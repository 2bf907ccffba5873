"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package writes INPUTS only: material tables evaluated on grids, voxel
phantoms, EPID layer stacks, spectra, fluence maps and response LUTs
(SURVEY.md section 8(c) "Cross-section / stopping-power tables" and 8(d)
"Configs as concrete synthetic inputs").  It contains none of the transport
method's arithmetic (no interpolation, no sampling, no tracking); the oracle
(`oracle/`) and the CUDA library (`paper_2510_24154_b200/csrc/`) each
implement that on their own and neither is imported here.
"""
from .tables import make_tables, MATERIALS, ELEMENTS  # noqa: F401
from .configs import make_config, head_config, CONFIG_NAMES  # noqa: F401
