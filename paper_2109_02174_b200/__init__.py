"""B200-native parallel-beam filtered back-projection (arxiv 2109.02174 hot path)."""
