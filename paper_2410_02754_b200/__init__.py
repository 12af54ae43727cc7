"""B200-native Chebyshev-filtered spinor H.X (arxiv 2410.02754 hot path): C-ABI library + thin binding."""
