"""B200-native motion-focus hot path (arxiv 2601.07154): thin Python binding over
the C-ABI library declared in include/mf.h.  Importing the package does not load
the CUDA library; the first call does, and fails loudly if it is missing."""
__version__ = "0.1.0"
