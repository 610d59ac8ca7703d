"""mkf — B200-native batched Kalman-filter track fitting and building (arxiv 2002.06295 hot path).

`paper_2002_06295_b200.binding` is the thin ctypes layer over the C-ABI library (include/mkf.h);
`paper_2002_06295_b200.datagen` makes the seeded synthetic events. Nothing here imports oracle/."""
