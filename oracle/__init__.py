"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT (see me_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Nothing here imports the CUDA package's kernels, generator or binding.
"""
from .me_oracle import (build, color_matrix, me_ggttx, me_eemumu, partial_amplitudes, matrix_elements,
                        su3_generators, DENOM, NGLUONS)  # noqa: F401
from . import selection  # noqa: F401,E402
