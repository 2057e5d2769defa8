"""paper_1208_0302_b200 — B200-native GA inversion of Milne-Eddington Stokes profiles (GENESIS hot path).

The product is the C-ABI library built from csrc/ (libme_b200.so; see include/me.h); `binding` is the thin
Python layer over it and `workloads` the seeded synthetic-input recipes.
"""
