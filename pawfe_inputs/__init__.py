"""Seeded synthetic inputs for the PAW-FE R-ChFSI filter path (arxiv/paper_2604_26037).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2604_26037_b200``).  It holds none of the method's arithmetic: no finite-element
matrices, no projector integrals, no operator applications, no filter.  It only produces the
*data* a PAW-FE calculation is given:

* the five workload shapes of BASELINE.json ``configs`` (+ reduced-cell "twins" for parity tests),
* atom positions (sequential rejection sampling, minimum-image separation >= 2 bohr),
* the synthetic pseudopotential "dataset": Gaussian well parameters (Z, sigma), the projector
  channel table (l, m, sigma, amplitude) with unit-L2-norm amplitudes, and the coupling
  matrices D (= Delta_H) and Delta_S,
* seeded random vector blocks.

The paper's own workloads (Pt clusters, Te/WS2, JTH PAW data) are not
available; these inputs stand in for them with the same shapes (Table 2 for (p, h)).
"""
from .configs import (  # noqa: F401
    Config,
    CONFIGS,
    get_config,
    twin,
    make_system,
    System,
    random_block,
    projector_table,
)
