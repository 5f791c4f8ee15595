"""B200-native direct incoherent dedispersion (arxiv/paper_1112_0065 hot path)."""
