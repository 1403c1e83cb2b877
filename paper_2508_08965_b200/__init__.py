"""B200-native CGKS-5 / S2O4 hot path (arxiv/paper_2508_08965).  See DESIGN.md."""
