"""B200-native leading-order matrix elements (the CUDACPP hot path of arxiv 2510.05392).

`inputs`  : seeded RAMBO momenta + parameter card (shared with the oracle, no physics).
`binding` : thin ctypes binding over the C-ABI in include/mg5_b200.h (argument marshalling only).
`gen`     : build-time process generator (Feynman diagrams, colour algebra, CUDA emission).
"""
