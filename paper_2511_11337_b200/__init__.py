"""B200-native (sm_100a) chunk-parallel neural range coder — the hot path of BOA Constrictor
(arXiv 2511.11337).  `paper_2511_11337_b200.boa` is the thin binding over the C ABI in
`include/boa.h`; `paper_2511_11337_b200.synth` holds the seeded input generators.

Nothing here imports `oracle/`: the product path fails loudly without the CUDA library.
"""
