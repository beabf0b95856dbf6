"""B200-native coupled FDTD-LLG hot path (arXiv 2103.12819): CUDA library + thin binding."""
from . import workloads  # noqa: F401
