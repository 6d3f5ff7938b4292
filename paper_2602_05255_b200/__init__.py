"""B200-native low-rank updates of determinants and Pfaffians (arxiv/paper_2602_05255).

``lrux``      ctypes binding of the C-ABI library (include/lrux.h)
``mc``        stream-ordered Metropolis chains (harness)
``workload``  seeded synthetic inputs (no method arithmetic)
``build``     nvcc build of lib/liblrux.so for sm_100a
"""
