"""B200-native CheFSI hot path (arxiv 2302.09708): C-ABI CUDA library + thin Python binding."""
__version__ = "0.1.0"
