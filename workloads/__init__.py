"""Seeded synthetic inputs shared by the oracle tests and the CUDA harness.
Holds no operator arithmetic: only random coefficients and closed-form mesh
geometry."""
