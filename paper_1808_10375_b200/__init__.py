"""B200-native multi-mode difference-map (DM) ptychography hot path (arXiv:1808.10375 Section II).

Import `paper_1808_10375_b200.dm` for the binding of the C-ABI library (include/dm.h);
`paper_1808_10375_b200.synth` holds the seeded input generators only.
"""
