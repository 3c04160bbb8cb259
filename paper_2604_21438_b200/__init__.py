"""B200-native hydro hot path of SFUMATO# (arxiv/paper_2604_21438): thin Python binding of libsfh.

Every step of the path runs in the CUDA kernels of csrc/ behind the C ABI of include/sfh.h; this
package only marshals arguments (torch is used for device memory and streams).  There is no CPU
fallback: importing works without a GPU (so that the ABI can be inspected), every compute call
needs one.
"""
from .binding import (Mesh, SfhError, load_library, library_path, declared_symbols, measure_fp64_rate, cfl_dt_noalloc,  # noqa: F401
                      N, NV, BLK)
