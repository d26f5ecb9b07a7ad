"""paper_2607_02584_b200 — B200-native RotateAttention hot path (hand-written CUDA for sm_100a behind a
C-ABI, include/rotattn.h).  Importing the package loads librotattn.so and fails loudly if it is missing."""
from . import binding  # noqa: F401
