"""B200-native lineal path function (arXiv 1601.04359): thin Python binding over the
C-ABI library in csrc/ (see include/lpf.h).  The CUDA library is loaded on first use and
its absence is an error -- there is no CPU fallback."""
