"""galario-b200: GALARIO hot path (arXiv:1709.06999) as hand-written sm_100a CUDA behind a C ABI."""
