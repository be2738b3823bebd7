"""B200-native FLARE B2 force-field hot path (arxiv 2204.12573): thin Python binding over the
C-ABI library libflare_b200.so (include/flare_b200.h).  Importing the package does not load the
library; the first call into `paper_2204_12573_b200.flare` does, and fails loudly if it is missing."""

__all__ = ["workloads"]
