"""tangram-b200: B200-native decode attention over a ragged, non-uniformly compressed KV cache
(Tangram, arxiv/paper_2606_06302).  `binding` is the thin ctypes layer over the C-ABI library
declared in include/tangram.h; `inputs` holds the seeded synthetic input generators."""
