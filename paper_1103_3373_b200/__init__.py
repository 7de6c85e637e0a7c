"""B200-native unsplit hydro patch-group solver (arXiv:1103.3373 hot path)."""
