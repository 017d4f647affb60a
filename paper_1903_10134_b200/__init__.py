"""B200-native mDPD velocity-Verlet timestep (arxiv/paper_1903_10134 hot path).

``csrc/mdpd_b200.cu`` holds the hand-written sm_100a kernels and the C-ABI of ``include/mdpd.h``;
``binding.py`` is the thin ctypes layer; ``build.py`` compiles the library in-tree with nvcc.
Importing the package never builds and never falls back to a CPU path.
"""
from .binding import (LIB_PATH, SYMBOLS, MdpdError, Simulation, build_flags, lib, make_params, mdpd_params,  # noqa: F401
                      probe_issue_rates)
from .build import build  # noqa: F401
