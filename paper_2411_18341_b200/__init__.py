"""B200-native RK4 hot path of PHOENIX (arXiv 2411.18341): C-ABI library + thin Python binding."""
