"""CPU oracle for the BOA Constrictor hot path (arXiv 2511.11337) — TEST INFRASTRUCTURE ONLY.

Plain, slow, fp64 / exact-integer numpy + pure-Python restatement of what the path computes,
written from PAPER.md (cited as P:<line>) with the readings listed in DESIGN.md §"Readings".
It shares no code with the CUDA path under `paper_2511_11337_b200/csrc/` and neither imports
the other.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import it; the product never routes through it.

Modules
  model.py       O1  Mamba-1 step function  (eq. 4-5; Alg. 1; eq. 16, 18-22 P:361-380)
  quantise.py    O2  softmax (eq. 6) and the strictly-positive integer table (eq. 7)
  rangecoder.py  O3  range encoder / decoder (eq. 8-13)
  container.py   O4  the .boa container
  codec.py            chunk-parallel compress / decompress

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md §"What pins the oracle".
Unpinned: the compressed BYTES of the model path are implementation-defined (they depend on
the last bits of the logits) — "parity unpinned" for that one quantity; everything that
produces them (step, quantiser, coder, container) is pinned separately.
"""
