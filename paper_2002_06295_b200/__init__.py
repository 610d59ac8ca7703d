"""mkf — B200-native batched Kalman-filter track fitting and building (arxiv 2002.06295 hot path).

`paper_2002_06295_b200.binding` is the thin ctypes layer over the C-ABI library (include/mkf.h) built from `csrc/`
by `paper_2002_06295_b200.build`. Nothing else lives here: the synthetic inputs and the parity metrics are in the
top-level `workloads/` package, the checker in `oracle/`; this package imports neither."""
