"""Seeded synthetic inputs (`datagen`) and the parity metrics (`parity`) shared by tests/ and bench.py.

Not part of the product package: the generator simulates a toy detector (its own numpy helix, Bethe-Bloch and Highland
for the *truth*), and the parity module holds the tolerances of BASELINE.json north_star. Neither is imported by
paper_2002_06295_b200/ or by oracle/."""
