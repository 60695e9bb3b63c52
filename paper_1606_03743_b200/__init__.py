"""B200-native (sm_100a) implementation of the hot path of arXiv 1606.03743: potential and field of
charged BEM triangles / rectangles by Gaussian cubature.  The product is the C-ABI CUDA library
`libbemcub.so` (include/bemcub.h); `bemcub` is its thin ctypes binding, `synth` the seeded input
generators shared with the tests' CPU oracle (no arithmetic of the method lives there)."""
