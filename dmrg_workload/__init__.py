"""Seeded synthetic input generators for the two-dot sigma-vector hot path.

This package builds the INPUTS of the hot path (integrals, block-sparse operator
store, operator-pair term list, trial vector).  It is shared by the CUDA path and
by the CPU oracle and therefore contains none of the hot path's arithmetic (no
sigma contraction, no Davidson); it imports neither `oracle` nor the CUDA package.
"""
