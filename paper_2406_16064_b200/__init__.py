"""B200-native LLG hot path (arxiv 2406.16064): thin Python binding over libmm.so (include/mm.h).

`from paper_2406_16064_b200 import Sim` needs the CUDA library and a GPU and fails loudly without
them; `paper_2406_16064_b200.workloads` (seeded inputs) is importable anywhere.
"""
from .binding import Sim, MMError, load_library, F32, F64, RK4, DOPRI5, CAYLEY_RK4, DMI_NONE, DMI_BULK, DMI_INTERFACIAL, DMI_D2D  # noqa: F401
