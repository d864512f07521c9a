"""helios_rt: B200-native (sm_100a) radiative-transfer step of THOR+HELIOS (arXiv 2203.02293).

`workloads` is importable without a GPU; the binding (`helios_rt`) loads the CUDA C-ABI library and
fails loudly if it is missing -- there is no CPU fallback.
"""
from .workloads import IMPROVED, NONISOTHERMAL, TOA_SPECTRUM  # noqa: F401
